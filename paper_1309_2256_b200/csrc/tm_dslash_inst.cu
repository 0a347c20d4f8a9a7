// tm_dslash_inst.cu -- one translation unit per (TM_PREC, TM_RECON), compiled with -DTM_PREC=.. -DTM_RECON=..
#include "tm_dslash.cuh"

#ifndef TM_PREC
#error "compile with -DTM_PREC={8,4,2} -DTM_RECON={18,12}"
#endif

namespace tmk {

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
    a.parity = p.out_parity;
    a.nrhs = p.nrhs;
    a.eps = p.dagger ? -1.0 : 1.0;
    for (int k = 0; k < 4; ++k) a.pq[k] = p.pq[k];
    const int n = p.nrhs;
    kernel_timing_begin(st);
#if TM_PREC == 8
    if (n % 2 == 0) launch_nr<TM_PREC, TM_RECON, 2>(a, n / 2, st);
    else launch_nr<TM_PREC, TM_RECON, 1>(a, n, st);
#else
    if (n % 3 == 0) launch_nr<TM_PREC, TM_RECON, 3>(a, n / 3, st);
    else if (n % 4 == 0) launch_nr<TM_PREC, TM_RECON, 4>(a, n / 4, st);
    else if (n % 2 == 0) launch_nr<TM_PREC, TM_RECON, 2>(a, n / 2, st);
    else launch_nr<TM_PREC, TM_RECON, 1>(a, n, st);
#endif
    kernel_timing_end(st);
    TM_LAUNCH_CHECK("dslash_kernel");
    return TM_OK;
}

} // namespace tmk
