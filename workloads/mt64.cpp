// Seeded uniform stream shared by the oracle tests and the CUDA-path tests (SURVEY.md §8(d),
// "Common conventions").  This file holds NO arithmetic of the AMG-DD method: it only turns a
// seed into the uniform draws u_k = (mt19937_64 draw >> 11) * 2^-53, taken in index order.
// Input generators are the one thing both sides may share (they see identical bytes).
#include <cstdint>
#include <random>

extern "C" {

// out[k] = k-th uniform in [0,1) of std::mt19937_64(seed), k = 0..n-1.
void wl_uniform(uint64_t seed, int64_t n, double* out) {
    std::mt19937_64 g(seed);
    for (int64_t k = 0; k < n; ++k) out[k] = (double)(g() >> 11) * 0x1.0p-53;
}

// raw 64-bit draws (used for the known-answer test of the generator and for top-bit decisions)
void wl_raw(uint64_t seed, int64_t n, uint64_t* out) {
    std::mt19937_64 g(seed);
    for (int64_t k = 0; k < n; ++k) out[k] = g();
}

}  // extern "C"
