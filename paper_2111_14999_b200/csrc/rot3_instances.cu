// rot3_instances.cu -- the instantiations of k_rotate_v3<KS, GB, MTW, MODE> (rotate_v3.cuh), split over four
// translation units by KS range (-DROT3_PART=0..3) so that build.py can compile them in parallel.
// pe_rot3_kernel_part<P>(KS, GB, MTW, mode) returns the kernel's host stub, or nullptr if KS is not in this part.
#include "rotate_v3.cuh"

#ifndef ROT3_PART
#error "compile with -DROT3_PART=0..3"
#endif

namespace {

template <int KS, int GB, int MTW>
const void* pick(int mode)
{
    if (mode == 0) return (const void*)pe::k_rotate_v3<KS, GB, MTW, 0>;
    if (mode == 1) return (const void*)pe::k_rotate_v3<KS, GB, MTW, 1>;
    return (const void*)pe::k_rotate_v3<KS, GB, MTW, 3>;
}

// GB per KS: the smallest that fills whole a5 column tiles (g0) or the largest whose accumulators fit (g1 for one
// tile of b2 per item, g2 for two); phoebe_elph.cu (rot3_min_gb / rot3_max_gb) picks among exactly these
template <int KS>
const void* kernel_ks(int GB, int MTW, int mode)
{
    constexpr int g0 = (KS == 1 || KS == 3) ? 2 : 1;
    constexpr int g1 = KS == 1 ? 8 : KS == 2 ? 4 : (KS == 3 || KS == 4) ? 2 : 1;
    constexpr int g2 = KS == 1 ? 4 : (KS == 2 || KS == 3) ? 2 : 1;
    if (MTW == 1) return GB == g1 ? pick<KS, g1, 1>(mode) : pick<KS, g0, 1>(mode);
    return GB == g2 ? pick<KS, g2, 2>(mode) : pick<KS, g0, 2>(mode);
}

}  // namespace

#define ROT3_CASE(K) case K: return kernel_ks<K>(GB, MTW, mode);

#if ROT3_PART == 0
extern "C" const void* pe_rot3_kernel_part0(int KS, int GB, int MTW, int mode)
{
    switch (KS) { ROT3_CASE(1) ROT3_CASE(2) default: return nullptr; }
}
#elif ROT3_PART == 1
extern "C" const void* pe_rot3_kernel_part1(int KS, int GB, int MTW, int mode)
{
    switch (KS) { ROT3_CASE(3) ROT3_CASE(4) ROT3_CASE(5) default: return nullptr; }
}
#elif ROT3_PART == 2
extern "C" const void* pe_rot3_kernel_part2(int KS, int GB, int MTW, int mode)
{
    switch (KS) { ROT3_CASE(6) ROT3_CASE(7) ROT3_CASE(8) ROT3_CASE(9) default: return nullptr; }
}
#else
extern "C" const void* pe_rot3_kernel_part3(int KS, int GB, int MTW, int mode)
{
    switch (KS) { ROT3_CASE(10) ROT3_CASE(11) ROT3_CASE(12) default: return nullptr; }
}
#endif
