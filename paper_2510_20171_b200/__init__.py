"""paper_2510_20171_b200 -- B200-native on-device data path of the NCCLX collectives
(AllToAllv with device-resident counts; fixed-order fp32 sum behind AllReduce /
ReduceScatter).  The product is csrc/ (sm_100a CUDA kernels behind the C ABI of
include/ncclx_b200.h); `binding` is its ctypes marshalling layer; `workloads` holds the
seeded synthetic input generators (no method arithmetic)."""
from . import binding, workloads  # noqa: F401
from .binding import *  # noqa: F401,F403
