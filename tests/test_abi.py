"""The C-ABI library builds, loads without a GPU and exports every symbol include/fhgs.h declares; the header is
plain C; the host-side validation (no device work) rejects bad arguments.  No compute call is made here."""
import ctypes
import os
import re
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "fhgs.h")


def _declared():
    src = open(HEADER).read()
    return sorted(set(re.findall(r"FHGS_API\s+[\w\s\*]+?\b(fhgs_\w+)\s*\(", src)))


def test_header_compiles_as_c(tmp_path):
    c = tmp_path / "t.c"
    c.write_text('#include "fhgs.h"\nint main(void) { fhgs_params p; (void)p; return (int)FHGS_OK; }\n')
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-c", str(c), "-o",
                    str(tmp_path / "t.o")], check=True)


def test_library_exports_every_declared_symbol():
    from paper_2505_19154_b200 import build
    lib = ctypes.CDLL(build.build())
    names = _declared()
    assert {"fhgs_project", "fhgs_bin_sort", "fhgs_render", "fhgs_fuse_features"} <= set(names)
    for nm in names:
        assert hasattr(lib, nm), nm
    from paper_2505_19154_b200 import binding
    assert sorted(binding.EXPORTS) == names
    lib.fhgs_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.fhgs_version()


def test_scratch_bytes_and_defaults_without_device():
    from paper_2505_19154_b200 import binding as fb
    p = fb.default_params()
    assert abs(p.z_near - 0.2) < 1e-7 and abs(p.alpha_max - 0.9999) < 1e-7 and abs(p.t_min - 1e-4) < 1e-10
    assert p.q_cutoff == 9.0 and abs(p.cov_dilation - 0.3) < 1e-7 and abs(p.jac_clamp - 1.3) < 1e-7
    fb.lib.fhgs_scratch_bytes.restype = ctypes.c_size_t
    a = fb.lib.fhgs_scratch_bytes(ctypes.c_int32(1000), ctypes.c_int32(64), ctypes.c_int32(64), ctypes.c_uint64(4096))
    b = fb.lib.fhgs_scratch_bytes(ctypes.c_int32(1000000), ctypes.c_int32(1920), ctypes.c_int32(1080), ctypes.c_uint64(40000000))
    assert 0 < a < b and a % 256 == 0 and b % 256 == 0
    assert fb.lib.fhgs_scratch_bytes(ctypes.c_int32(-1), ctypes.c_int32(64), ctypes.c_int32(64), ctypes.c_uint64(0)) == 0
