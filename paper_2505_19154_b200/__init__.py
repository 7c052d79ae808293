"""FHGS hot path for B200 (sm_100a): projection, tile binning + onesweep sort, compositing of
RGB + D feature channels, and weight-aggregated feature fusion behind a C ABI (include/fhgs.h).

`inputs` (seeded synthetic generators) is importable without the CUDA extension; `binding`
loads libfhgs.so and fails loudly if it is missing -- there is no CPU fallback."""
