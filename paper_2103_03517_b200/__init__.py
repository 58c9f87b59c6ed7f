"""B200-native checkerboard Metropolis for classical Heisenberg spins (arXiv 2103.03517): the hot path behind a C ABI.

`binding` -- ctypes layer over libmc_b200.so (include/mc.h); `build` -- nvcc build of the library; `inputs` -- seeded
synthetic inputs (no method arithmetic); `replicas` -- independent points over several GPUs; `configs` -- the BASELINE.json
workloads; `analysis` -- host-side fits.  There is no CPU fallback and nothing here imports the oracle.
"""
__all__ = ["analysis", "binding", "build", "configs", "inputs", "replicas"]
