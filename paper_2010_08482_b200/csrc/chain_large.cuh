// Large-sector chain kernel (sectors whose carried panel does not fit in shared memory) -- placeholder, see chain.cuh.
#pragma once
#include "chain.cuh"

namespace ctqmc {
inline int large_configure(const DevImp&, int, int*, size_t*, int*) { return -4; }
inline int large_ensure_scratch(const DevImp&, int, int, double**, size_t*) { return -4; }
inline int large_enqueue(const ChainParams&, int, size_t, int, double*, cudaStream_t) { return -4; }
}  // namespace ctqmc
