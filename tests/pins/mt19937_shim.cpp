// TEST-ONLY pin: the C++ standard library's std::mt19937 is MT19937 seeded by init_genrand (the standard fixes its
// 10000th value from the default seed 5489 as 4123659995).  Exposed through C symbols for ctypes.
#include <cstdint>
#include <random>

extern "C" void pin_mt19937_sequence(uint32_t seed, uint32_t count, uint32_t* out)
{
    std::mt19937 g(seed);
    for (uint32_t k = 0; k < count; ++k) out[k] = (uint32_t)g();
}
