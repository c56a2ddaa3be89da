"""B200-native direct N-body force / jerk / potential (after arxiv 0707.0438, "kirin").

Only what the hot path needs lives here:
  inputs.py   seeded synthetic workloads (no method arithmetic)
  binding.py  thin ctypes marshalling over the C-ABI library (include/nbk.h)
  sharded.py  opt-in j-sharding over several GPUs (C-ABI calls + two all-reduces)
  build.py    nvcc build of csrc/ -> libnbk.so (sm_100a)
  csrc/       CUDA kernels + C-ABI + host Hermite driver
The CUDA library is loaded lazily by `binding`; importing this package or
`inputs` does not need a GPU.
"""
__all__ = ["inputs", "binding", "build"]
