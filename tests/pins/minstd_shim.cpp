// TEST-ONLY pin: the C++ standard library's std::minstd_rand0 IS the generator of PAPER.md:170 Eq. 7
// (multiplier 16807, modulus 2^31-1, increment 0).  Exposed through C symbols for ctypes.
#include <cstdint>
#include <random>

extern "C" void pin_minstd_rand0_sequence(uint32_t seed_state, uint32_t count, uint32_t* out)
{
    std::minstd_rand0 g(seed_state);
    for (uint32_t k = 0; k < count; ++k) out[k] = (uint32_t)g();
}

extern "C" uint32_t pin_minstd_rand0_discard(uint32_t seed_state, uint64_t n)
{
    std::minstd_rand0 g(seed_state);
    g.discard(n);
    return (uint32_t)g();
}
