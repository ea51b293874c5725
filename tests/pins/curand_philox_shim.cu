// TEST-ONLY pin: exposes NVIDIA cuRAND's own Philox4x32-10 block function (the host branch of
// curand_philox4x32_x.h, shipped with the CUDA toolkit) through a C symbol, so that the oracle's
// Philox can be compared with an implementation neither side of this repo wrote.
// Built by tests/pins/build_pins.py with nvcc (host code only; no GPU needed).
#define QUALIFIERS static inline __host__ __device__
#include <cuda_runtime.h>
#include <curand_philox4x32_x.h>

extern "C" void pin_curand_philox4x32_10(const unsigned int ctr[4], const unsigned int key[2], unsigned int out[4])
{
    uint4 c = make_uint4(ctr[0], ctr[1], ctr[2], ctr[3]);
    uint2 k = make_uint2(key[0], key[1]);
    uint4 r = curand_Philox4x32_10(c, k);
    out[0] = r.x; out[1] = r.y; out[2] = r.z; out[3] = r.w;
}
