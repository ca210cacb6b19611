// tests/pins/curand_philox_shim.cpp -- TEST PIN, not product code.
// Exposes two LIBRARY routines of the CUDA toolkit so that the oracle's own
// Philox4x32-10 (oracle/muca_oracle.cpp) can be checked against something
// other than itself (PAPER.md:107 names the generator, Ref. [41]):
//   pin_curand_philox4x32_10 : the toolkit's device routine
//       curand_Philox4x32_10(uint4 ctr, uint2 key)  (curand_philox4x32_x.h),
//       compiled for the host by redefining QUALIFIERS;
//   pin_curand_host_generate : libcurand's HOST generator
//       CURAND_RNG_PSEUDO_PHILOX4_32_10 (needs no GPU).
// Build: g++ -O1 -shared -fPIC -I$CUDA/include shim.cpp -L$CUDA/lib64 -lcurand
#include <cstdint>
#include <vector_types.h>
#define QUALIFIERS static inline
#include <curand_philox4x32_x.h>
#undef QUALIFIERS
#include <curand.h>

extern "C" {

void pin_curand_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
    uint4 c; c.x = ctr[0]; c.y = ctr[1]; c.z = ctr[2]; c.w = ctr[3];
    uint2 k; k.x = key[0]; k.y = key[1];
    const uint4 r = curand_Philox4x32_10(c, k);
    out[0] = r.x; out[1] = r.y; out[2] = r.z; out[3] = r.w;
}

// n 32-bit outputs of the host generator with the given seed and offset.
int pin_curand_host_generate(unsigned long long seed, unsigned long long offset, uint32_t* out, size_t n) {
    curandGenerator_t g;
    if (curandCreateGeneratorHost(&g, CURAND_RNG_PSEUDO_PHILOX4_32_10) != CURAND_STATUS_SUCCESS) return -1;
    int rc = 0;
    if (curandSetPseudoRandomGeneratorSeed(g, seed) != CURAND_STATUS_SUCCESS) rc = -2;
    if (!rc && curandSetGeneratorOffset(g, offset) != CURAND_STATUS_SUCCESS) rc = -3;
    if (!rc && curandGenerate(g, out, n) != CURAND_STATUS_SUCCESS) rc = -4;
    curandDestroyGenerator(g);
    return rc;
}

// n uniform floats of the host generator with the given seed and offset: the library's own mapping of the raw 32-bit
// words (pin_curand_host_generate with the same seed and offset) to (0, 1] -- pins the oracle's uniform32 (R23).
int pin_curand_host_generate_uniform(unsigned long long seed, unsigned long long offset, float* out, size_t n) {
    curandGenerator_t g;
    if (curandCreateGeneratorHost(&g, CURAND_RNG_PSEUDO_PHILOX4_32_10) != CURAND_STATUS_SUCCESS) return -1;
    int rc = 0;
    if (curandSetPseudoRandomGeneratorSeed(g, seed) != CURAND_STATUS_SUCCESS) rc = -2;
    if (!rc && curandSetGeneratorOffset(g, offset) != CURAND_STATUS_SUCCESS) rc = -3;
    if (!rc && curandGenerateUniform(g, out, n) != CURAND_STATUS_SUCCESS) rc = -4;
    curandDestroyGenerator(g);
    return rc;
}

}  // extern "C"
