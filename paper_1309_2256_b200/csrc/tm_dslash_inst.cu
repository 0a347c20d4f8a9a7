// tm_dslash_inst.cu -- one translation unit per (TM_PREC, TM_RECON), compiled with -DTM_PREC=.. -DTM_RECON=..
#include "tm_dslash_tile.cuh"
#include <cstdlib>

#ifndef TM_PREC
#error "compile with -DTM_PREC={8,4,2} -DTM_RECON={18,12}"
#endif

#ifndef TM_LC_RB
#define TM_LC_RB 12
#endif
#ifndef TM_LC_MINB
#define TM_LC_MINB 2
#endif
#ifndef TM_LC_TPC
#define TM_LC_TPC 16
#endif

namespace tmk {

template <int PREC, int RECON>
int link_cache_build_t(const Geo& g, const void* gauge, void* cache, cudaStream_t st);

template <>
int launch_dslash_t<TM_PREC, TM_RECON>(const Geo& g, const DslashParams& p, cudaStream_t st)
{
    DslashKArgs a;
    a.g = g;
    a.gauge = static_cast<const char*>(p.gauge);
    a.out = static_cast<char*>(p.out);
    a.in = static_cast<const char*>(p.in);
    a.x = static_cast<const char*>(p.x);
    a.link_block = link_block_bytes(g, TM_PREC, TM_RECON);
    a.stride_out = p.rhs_stride_out;
    a.stride_in = p.rhs_stride_in;
    a.stride_x = p.rhs_stride_x;
    a.active = p.active;
    a.link_cache = static_cast<const char*>(p.link_cache);
    a.dot_with = static_cast<const char*>(p.dot_with);
    a.stride_dot = p.dot_stride;
    a.dot_partial = p.dot_partial;
    a.axpy_y = static_cast<const char*>(p.axpy_y);
    a.stride_y = p.axpy_y_stride;
    a.axpy_coef = static_cast<const char*>(p.axpy_coef);
    a.stride_coef = p.axpy_coef_stride;
    a.parity = p.out_parity;
    a.nrhs = p.nrhs;
    a.eps = p.dagger ? -1.0 : 1.0;
    for (int k = 0; k < 4; ++k) a.pq[k] = p.pq[k];
    const int n = p.nrhs;
#if TM_RECON >= 200
    if (n != 1) return TM_ERR_ARG; // before the timing bracket opens (launch_dslash sends nrhs > 1 to the plain instantiations)
#endif
    kernel_timing_begin(st);
#if TM_RECON >= 200
    // temporal gauge declared (tm.h): the single-rhs kernel that loads no link for temporal hops inside the lattice
    launch_tile<TM_PREC, TM_RECON, 128, 1, 4, 0>(a, p.dagger != 0, st);
#elif TM_PREC == 8
    // fp64: one thread per (site, rhs); threads of one site share the link lines in L1 (measured faster than two rhs per
    // thread at 128 registers)
    launch_nr<TM_PREC, TM_RECON, 1>(a, n, st);
#else
    // Launch shapes from the B200 sweeps ("Optimisation log"):
    //   1 rhs      128 sites per CTA, links per thread, packed fma.rn.f32x2 arithmetic, 4 CTAs/SM (128 registers)
    //   2..4 rhs   32 sites x 4 rhs, links of the tile built in shared memory, 6 CTAs/SM
    //   5..6 rhs   32 sites x 6 rhs, 4 CTAs/SM
    //   > 6 rhs    32 sites x 12 rhs, 2 CTAs/SM (80 registers); inside a solve the tile images come from the link cache
    //              by cp.async.bulk, 16 tiles per CTA (7..8 rhs: 32 sites x 8 rhs, 3 CTAs/SM).  Tiles per CTA at 32^3x64: fp16
    //              storage flat from 2 to 16 (332 solves/s), fp32 storage 237 / 242 / 248 solves/s at 4 / 8 / 16; 32 and more lose to the tail
    const bool dg = p.dagger != 0;
    if (n == 1) launch_tile<TM_PREC, TM_RECON, 128, 1, 4, 0>(a, dg, st);
    else if (n <= 4) launch_tile<TM_PREC, TM_RECON, 32, 4, 6, 1>(a, dg, st);
    else if (n <= 6) launch_tile<TM_PREC, TM_RECON, 32, 6, 4, 1>(a, dg, st);
#ifdef TM_SWEEP
    // probe builds only (_work/): the launch shape of the link-cache kernel is picked by the environment at run time
    else if (a.link_cache) {
        static const int cfg = getenv("TM_LC_CFG") ? atoi(getenv("TM_LC_CFG")) : 0;
        switch (cfg) {
#define TM_CASE(id, RB, MINB, TPC) case id: launch_tile_lc<TM_PREC, TM_RECON, RB, MINB, TPC>(a, dg, st); break;
            TM_SWEEP_CASES
#undef TM_CASE
        default: launch_tile_lc<TM_PREC, TM_RECON, 12, 2, 4>(a, dg, st);
        }
    }
#else
    // 7 or 8 right-hand sides (the last batch of 200 sources, the paper's N_HP = 8): CTAs of 8 warps at 3 per SM instead of 12-warp
    // CTAs with a third of their warps idle (8 rhs at 32^3x64: 0.533 -> 0.480 ms per launch, 287 -> 312 solves/s)
    else if (a.link_cache && n <= 8) launch_tile_lc<TM_PREC, TM_RECON, 8, 3, TM_LC_TPC>(a, dg, st);
    else if (a.link_cache) launch_tile_lc<TM_PREC, TM_RECON, TM_LC_RB, TM_LC_MINB, TM_LC_TPC>(a, dg, st);
#endif
    else launch_tile<TM_PREC, TM_RECON, 32, 12, 2, 1>(a, dg, st);
#endif
    kernel_timing_end(st);
    TM_LAUNCH_CHECK("dslash_kernel");
    return TM_OK;
}

#if TM_PREC == 2 && TM_RECON == 12
// template signature of the kernel that dominates the TSM step (12 rhs, fp16 storage, 12-real links): bench.py ties the
// DRAM traffic it quotes from an ncu capture to this string (tm_kernel_signature)
#define TM_STR2(x) #x
#define TM_STR(x) TM_STR2(x)
const char* lc_kernel_signature()
{
    return "dslash_tile_lc_kernel<prec=2,recon=12,RB=" TM_STR(TM_LC_RB) ",MINB=" TM_STR(TM_LC_MINB) ",TPC=" TM_STR(TM_LC_TPC) ">";
}
#endif

#if TM_PREC != 8 && TM_RECON < 200
template <>
int link_cache_build_t<TM_PREC, TM_RECON>(const Geo& g, const void* gauge, void* cache, cudaStream_t st)
{
    DslashKArgs a = {};
    a.g = g;
    a.gauge = static_cast<const char*>(gauge);
    a.link_block = link_block_bytes(g, TM_PREC, TM_RECON);
    launch_link_cache<TM_PREC, TM_RECON>(a, static_cast<char*>(cache), st);
    TM_LAUNCH_CHECK("link_cache_kernel");
    return TM_OK;
}
#endif

} // namespace tmk
