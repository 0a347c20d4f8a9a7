// tm_dslash_inst.cu -- one translation unit per (TM_PREC, TM_RECON), compiled with -DTM_PREC=.. -DTM_RECON=..
#include "tm_dslash_tile.cuh"
#include <cstdlib>

#ifndef TM_PREC
#error "compile with -DTM_PREC={8,4,2} -DTM_RECON={18,12}"
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
    kernel_timing_begin(st);
#if TM_PREC == 8
    static const int cfg64 = getenv("TM_DSLASH_F64_NR") ? atoi(getenv("TM_DSLASH_F64_NR")) : 1; // measured: one rhs per thread (links shared through L1) beats two at 128 registers
    if (n % 2 == 0 && cfg64 == 2) launch_nr<TM_PREC, TM_RECON, 2>(a, n / 2, st);
    else launch_nr<TM_PREC, TM_RECON, 1>(a, n, st);
#else
    // Launch shapes from the B200 sweep; the environment knobs exist for re-tuning:
    //   TM_DSLASH_SINGLE: 0 = 128 registers + prefetch, 1 = 128 registers (default), 2 = 96 registers + prefetch, -1 = dslash_kernel
    //   TM_DSLASH_MULTI : 0 = by nrhs (12 / 6 / 4 right-hand sides per CTA at 80 registers), 1 = 12 + prefetch, -1 = dslash_kernel
    static const int cfg_multi = getenv("TM_DSLASH_MULTI") ? atoi(getenv("TM_DSLASH_MULTI")) : 0;
    static const int cfg_single = getenv("TM_DSLASH_SINGLE") ? atoi(getenv("TM_DSLASH_SINGLE")) : 1;
    const bool dg = p.dagger != 0;
    if (n == 1) {
        switch (cfg_single) {
        case 0: launch_tile<TM_PREC, TM_RECON, 128, 1, 4, 0, true>(a, dg, st); break;
        case 1: launch_tile<TM_PREC, TM_RECON, 128, 1, 4, 0, false>(a, dg, st); break;
        case 2: launch_tile<TM_PREC, TM_RECON, 128, 1, 5, 0, true>(a, dg, st); break;
        default: launch_nr<TM_PREC, TM_RECON, 1>(a, n, st);
        }
    } else if (cfg_multi == 0) {
        if (n <= 4) launch_tile<TM_PREC, TM_RECON, 32, 4, 6, 1, false>(a, dg, st);
        else if (n <= 6) launch_tile<TM_PREC, TM_RECON, 32, 6, 4, 1, false>(a, dg, st);
        else if (a.link_cache) {
            static const int tpc = getenv("TM_DSLASH_TPC") ? atoi(getenv("TM_DSLASH_TPC")) : 4;
            static const int lcv = getenv("TM_DSLASH_LC") ? atoi(getenv("TM_DSLASH_LC")) : 0;
            if (lcv == 1) launch_tile_lc<TM_PREC, TM_RECON, 6, 5, 4>(a, dg, st);
            else if (lcv == 2) launch_tile_lc<TM_PREC, TM_RECON, 4, 8, 4>(a, dg, st);
            else if (lcv == 3) launch_tile_lc<TM_PREC, TM_RECON, 6, 4, 4>(a, dg, st);
            else if (tpc == 2) launch_tile_lc<TM_PREC, TM_RECON, 12, 2, 2>(a, dg, st);
            else if (tpc == 8) launch_tile_lc<TM_PREC, TM_RECON, 12, 2, 8>(a, dg, st);
            else launch_tile_lc<TM_PREC, TM_RECON, 12, 2, 4>(a, dg, st);
        }
        else launch_tile<TM_PREC, TM_RECON, 32, 12, 2, 1, false>(a, dg, st);
    } else if (cfg_multi == 1) {
        launch_tile<TM_PREC, TM_RECON, 32, 12, 2, 1, true>(a, dg, st);
    } else {
        if (n % 3 == 0) launch_nr<TM_PREC, TM_RECON, 3>(a, n / 3, st);
        else if (n % 4 == 0) launch_nr<TM_PREC, TM_RECON, 4>(a, n / 4, st);
        else if (n % 2 == 0) launch_nr<TM_PREC, TM_RECON, 2>(a, n / 2, st);
        else launch_nr<TM_PREC, TM_RECON, 1>(a, n, st);
    }
#endif
    kernel_timing_end(st);
    TM_LAUNCH_CHECK("dslash_kernel");
    return TM_OK;
}

#if TM_PREC != 8
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
