// Host-only check of the SMEM engine's shared-memory plan (tests/test_abi.py compiles and runs it with nvcc; no GPU
// needed): the state of the longest sequence of BASELINE.json configs[3] (n = 700, q = 8) has to fit one SM, regions
// must not overlap and must keep their alignment, max_n must be the exact limit.
#include <cstdio>
#include <new>
#include "../paper_1307_7820_b200/csrc/smem_engine.cuh"

template <int Q>
static int check()
{
    using C = smemseq::Cfg<Q>;
    const unsigned pool = C::MAX_SMEM - C::FIXED_BYTES;
    const int lim = smemseq::max_n<Q>();
    if (smemseq::make_layout<Q>(lim).total > pool || smemseq::make_layout<Q>(lim + Q).total <= pool) return 1;
    for (int n = 0; n <= lim; n += 7) {
        const smemseq::Layout L = smemseq::make_layout<Q>(n);
        const unsigned o[] = {L.W, L.X, L.val, L.wdh, L.dq, L.pm, L.rl, L.code, L.plan, L.flags, L.total};
        for (int i = 0; i + 1 < 11; ++i) if (o[i] > o[i + 1] || o[i] % 16) return 2;
        const unsigned NB = n / Q + 1;
        if (L.X - L.W < 4u * Q * NB * (NB - 1) / 2 || L.val - L.X < 2u * Q * NB * (NB + 1) / 2) return 3;
        if (n > 0 && L.total < smemseq::make_layout<Q>(n - 1).total) return 4;
    }
    std::printf("q=%d max_n=%d\n", Q, lim);
    return 0;
}

int main()
{
    if (check<4>() || check<5>() || check<6>() || check<7>() || check<8>()) return 1;
    if (smemseq::max_n<8>() < 700) return 2;                       // config 4 must run on this engine
    std::printf("smem_layout_check ok\n");
    return 0;
}
