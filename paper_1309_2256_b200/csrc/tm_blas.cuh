// tm_blas.cuh -- a5 of SURVEY.md 8(a): fused CG vector kernels with device-resident scalars.
//
// Every kernel touches each vector once, works on one-parity packed spinors [rhs] with explicit per-vector
// rhs strides (bytes), skips right-hand sides whose `active` flag is 0, and -- where it reduces -- uses a
// fixed-order reduction: warp shuffles -> shared memory -> one fp64 partial per block -> the last block to
// finish (ticket counter) sums the partials in index order and updates the per-rhs scalars.  No floating-point
// atomics, so a given input gives bit-identical scalars run to run and batched == unbatched.
#pragma once
#include "tm_layout.cuh"

namespace tmk {

constexpr int BLAS_THREADS = 256;
constexpr int BLAS_MAX_BLOCKS = 1184; // 148 SMs x 8

// per right-hand-side CG scalars, resident on the device
struct CgScal {
    double rr;      // |r_k|^2 (iterated)
    double rr_new;
    double pAp;
    double alpha, beta;
    double b2;      // |b''|^2
    double tol2;    // tol^2
    double aux;     // scratch result of plain norm2/dot reductions
    int iter;
    int max_iter;
    int status;     // tm_status
    int alpha_iter; // iteration (0-based) whose <p,Ap> produced `alpha`: update_xp applies x += alpha p only for that one
};

struct BlasCtx {
    CgScal* scal;            // [nrhs]
    unsigned char* active;   // [nrhs]
    double* partials;        // [nrhs][BLAS_MAX_BLOCKS]
    unsigned int* tickets;   // [nrhs]
};

enum { FIN_AUX = 0, FIN_PAP = 1, FIN_RR = 2, FIN_INIT = 3 };

// block-wide sum of `v` (all threads call); result valid in thread 0
template <int THREADS = BLAS_THREADS>
__device__ __forceinline__ double block_sum(double v)
{
    __shared__ double sm[THREADS / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __syncthreads(); // protect sm reuse across calls
    if (lane == 0) sm[warp] = v;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x < 32) {
        s = (threadIdx.x < THREADS / 32) ? sm[threadIdx.x] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    }
    return s;
}

// what a finished reduction means for the per-rhs CG scalars (one thread)
template <int FIN>
__device__ __forceinline__ void finish_scalar(const BlasCtx& c, int rhs, double tot)
{
    CgScal& s = c.scal[rhs];
    if (FIN == FIN_AUX) {
        s.aux = tot;
    } else if (FIN == FIN_INIT) { // tot = |b''|^2 : start of a solve
        s.b2 = tot;
        s.rr = tot;
        if (!(tot > 0.0)) c.active[rhs] = 0; // zero source: x = 0 is the solution
        if (!(tot == tot)) s.status = TM_ERR_BREAKDOWN; // NaN in the source
    } else if (FIN == FIN_PAP) {
        s.pAp = tot;
        s.alpha_iter = s.iter;
        if (!(tot > 0.0)) { // breakdown or NaN
            s.status = TM_ERR_BREAKDOWN;
            s.alpha = 0.0;
            c.active[rhs] = 0;
        } else {
            s.alpha = s.rr / tot;
        }
    } else { // FIN_RR: tot = |r_{k+1}|^2
        s.rr_new = tot;
        s.beta = tot / s.rr;
        s.rr = tot;
        s.iter += 1;
        if (tot <= s.tol2 * s.b2) {
            c.active[rhs] = 0;
            s.status = TM_OK;
        } else if (s.iter >= s.max_iter) {
            c.active[rhs] = 0;
            s.status = TM_ERR_MAXITER;
        } else if (!(tot == tot)) {
            c.active[rhs] = 0;
            s.status = TM_ERR_BREAKDOWN;
        }
    }
}

// two-stage deterministic reduction + scalar update by the last block of this rhs
template <int FIN>
__device__ __forceinline__ void reduce_finalize(const BlasCtx& c, int rhs, double local)
{
    const double bs = block_sum(local);
    __shared__ bool last;
    if (threadIdx.x == 0) {
        c.partials[(size_t)rhs * BLAS_MAX_BLOCKS + blockIdx.x] = bs;
        __threadfence();
        const unsigned int t = atomicAdd(&c.tickets[rhs], 1u);
        last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    double v = 0.0;
    const volatile double* p = c.partials + (size_t)rhs * BLAS_MAX_BLOCKS;
    // fixed order: thread k sums partials k, k+BLAS_THREADS, ... then the block tree
    for (int b = threadIdx.x; b < (int)gridDim.x; b += BLAS_THREADS) v += p[b];
    const double tot = block_sum(v);
    if (threadIdx.x == 0) {
        finish_scalar<FIN>(c, rhs, tot);
        c.tickets[rhs] = 0;
    }
}

struct VecArg {
    char* p;
    size_t stride; // bytes between right-hand sides
};

// out = (c0 + i c1 g5) in
template <int PREC>
__global__ void __launch_bounds__(BLAS_THREADS) twist_kernel(int Vh, VecArg out, VecArg in, double c0, double c1)
{
    typedef typename Prec<PREC>::real real;
    const int rhs = blockIdx.y;
    for (int cb = blockIdx.x * BLAS_THREADS + threadIdx.x; cb < Vh; cb += gridDim.x * BLAS_THREADS) {
        real v[24], o[24];
        load_spinor<PREC>(in.p + rhs * in.stride, Vh, cb, v);
#pragma unroll
        for (int k = 0; k < 12; ++k) {
            const real s5 = (k < 6) ? real(1) : real(-1);
            o[2 * k] = (real)c0 * v[2 * k] - s5 * (real)c1 * v[2 * k + 1];
            o[2 * k + 1] = (real)c0 * v[2 * k + 1] + s5 * (real)c1 * v[2 * k];
        }
        store_spinor<PREC>(out.p + rhs * out.stride, Vh, cb, o);
    }
}

// out(PO) = in(PI), optionally also out2(PO) = in  (r and p from r_hp)
template <int PO, int PI>
__global__ void __launch_bounds__(BLAS_THREADS) convert_kernel(int Vh, VecArg out, VecArg out2, VecArg in)
{
    typedef typename Prec<PI>::real ri;
    typedef typename Prec<PO>::real ro;
    const int rhs = blockIdx.y;
    for (int cb = blockIdx.x * BLAS_THREADS + threadIdx.x; cb < Vh; cb += gridDim.x * BLAS_THREADS) {
        ri v[24];
        ro o[24];
        load_spinor<PI>(in.p + rhs * in.stride, Vh, cb, v);
#pragma unroll
        for (int k = 0; k < 24; ++k) o[k] = (ro)v[k];
        store_spinor<PO>(out.p + rhs * out.stride, Vh, cb, o);
        if (out2.p) store_spinor<PO>(out2.p + rhs * out2.stride, Vh, cb, o);
    }
}

// |v|^2 -> FIN (FIN_AUX or FIN_INIT)
template <int PREC, int FIN>
__global__ void __launch_bounds__(BLAS_THREADS) norm2_kernel(int Vh, VecArg v_, BlasCtx c)
{
    typedef typename Prec<PREC>::real real;
    const int rhs = blockIdx.y;
    double acc = 0.0;
    for (int cb = blockIdx.x * BLAS_THREADS + threadIdx.x; cb < Vh; cb += gridDim.x * BLAS_THREADS) {
        real v[24];
        load_spinor<PREC>(v_.p + rhs * v_.stride, Vh, cb, v);
        real s = 0;
#pragma unroll
        for (int k = 0; k < 24; ++k) s = fma(v[k], v[k], s);
        acc += (double)s;
    }
    reduce_finalize<FIN>(c, rhs, acc);
}

// pAp = Re<p, Ap>; alpha = rr / pAp
template <int PREC>
__global__ void __launch_bounds__(BLAS_THREADS) dot_pAp_kernel(int Vh, VecArg p_, VecArg Ap_, BlasCtx c)
{
    typedef typename Prec<PREC>::real real;
    const int rhs = blockIdx.y;
    if (!c.active[rhs]) return;
    double acc = 0.0;
    for (int cb = blockIdx.x * BLAS_THREADS + threadIdx.x; cb < Vh; cb += gridDim.x * BLAS_THREADS) {
        real p[24], q[24];
        load_spinor<PREC>(p_.p + rhs * p_.stride, Vh, cb, p);
        load_spinor<PREC>(Ap_.p + rhs * Ap_.stride, Vh, cb, q);
        real s = 0;
#pragma unroll
        for (int k = 0; k < 24; ++k) s = fma(p[k], q[k], s);
        acc += (double)s;
    }
    reduce_finalize<FIN_PAP>(c, rhs, acc);
}

// x += alpha p; r -= alpha Ap; rr_new = |r|^2; beta, convergence
template <int PREC>
__global__ void __launch_bounds__(BLAS_THREADS) update_xr_kernel(int Vh, VecArg x_, VecArg r_, VecArg p_, VecArg Ap_, BlasCtx c)
{
    typedef typename Prec<PREC>::real real;
    const int rhs = blockIdx.y;
    if (!c.active[rhs]) return;
    const real alpha = (real)c.scal[rhs].alpha;
    double acc = 0.0;
    for (int cb = blockIdx.x * BLAS_THREADS + threadIdx.x; cb < Vh; cb += gridDim.x * BLAS_THREADS) {
        real x[24], r[24], p[24], q[24];
        load_spinor<PREC>(x_.p + rhs * x_.stride, Vh, cb, x);
        load_spinor<PREC>(p_.p + rhs * p_.stride, Vh, cb, p);
        load_spinor<PREC>(r_.p + rhs * r_.stride, Vh, cb, r);
        load_spinor<PREC>(Ap_.p + rhs * Ap_.stride, Vh, cb, q);
        real s = 0;
#pragma unroll
        for (int k = 0; k < 24; ++k) {
            x[k] = fma(alpha, p[k], x[k]);
            r[k] = fma(-alpha, q[k], r[k]);
            s = fma(r[k], r[k], s);
        }
        store_spinor<PREC>(x_.p + rhs * x_.stride, Vh, cb, x);
        store_spinor<PREC>(r_.p + rhs * r_.stride, Vh, cb, r);
        acc += (double)s;
    }
    reduce_finalize<FIN_RR>(c, rhs, acc);
}

// p = r + beta p
template <int PREC>
__global__ void __launch_bounds__(BLAS_THREADS) update_p_kernel(int Vh, VecArg p_, VecArg r_, BlasCtx c)
{
    typedef typename Prec<PREC>::real real;
    const int rhs = blockIdx.y;
    if (!c.active[rhs]) return;
    const real beta = (real)c.scal[rhs].beta;
    for (int cb = blockIdx.x * BLAS_THREADS + threadIdx.x; cb < Vh; cb += gridDim.x * BLAS_THREADS) {
        real r[24], p[24];
        load_spinor<PREC>(r_.p + rhs * r_.stride, Vh, cb, r);
        load_spinor<PREC>(p_.p + rhs * p_.stride, Vh, cb, p);
#pragma unroll
        for (int k = 0; k < 24; ++k) p[k] = fma(beta, p[k], r[k]);
        store_spinor<PREC>(p_.p + rhs * p_.stride, Vh, cb, p);
    }
}

// y(PY) = a*y + b*x(PX)  [+ |y|^2 -> aux if REDUCE]   (x_hp += x_lp ; r = b - Ax with a=-1,b=1 on y=Ax, x=b)
template <int PY, int PX, int REDUCE>
__global__ void __launch_bounds__(BLAS_THREADS) axpby_kernel(int Vh, VecArg y_, VecArg x_, double a, double b, BlasCtx c)
{
    typedef typename Prec<PY>::real ry;
    typedef typename Prec<PX>::real rx;
    const int rhs = blockIdx.y;
    double acc = 0.0;
    for (int cb = blockIdx.x * BLAS_THREADS + threadIdx.x; cb < Vh; cb += gridDim.x * BLAS_THREADS) {
        ry y[24];
        rx x[24];
        load_spinor<PY>(y_.p + rhs * y_.stride, Vh, cb, y);
        load_spinor<PX>(x_.p + rhs * x_.stride, Vh, cb, x);
        ry s = 0;
#pragma unroll
        for (int k = 0; k < 24; ++k) {
            y[k] = (ry)a * y[k] + (ry)b * (ry)x[k];
            s = fma(y[k], y[k], s);
        }
        store_spinor<PY>(y_.p + rhs * y_.stride, Vh, cb, y);
        acc += (double)s;
    }
    if (REDUCE) reduce_finalize<FIN_AUX>(c, rhs, acc);
}

// ---- fused truncated-CG iteration (LP mode) ------------------------------------------------------------------------
//   <p,Ap> = |M_pc p|^2 and |r|^2 come out of dslash epilogues as per-warp partials (warp_dot_store, tm_dslash.cuh), the
//   residual update r -= alpha A p happens in the epilogue that produces A p (fused_axpy); dot_finalize_kernel sums the
//   partials in a fixed order -> alpha / beta, convergence;  update_xp: x += alpha p, p = r + beta p (5 vector passes).

// tot[rhs] = sum_g partial[rhs][g] (fixed order), then the FIN scalar update (FIN_PAP or FIN_RR).  grid = nrhs blocks
constexpr int FIN_THREADS = 1024; // one CTA per rhs sums 32 768 partials at 32^3 x 64: latency-bound, so many threads and loads in flight
template <int FIN>
__global__ void __launch_bounds__(FIN_THREADS) dot_finalize_kernel(const double* partial, int ngroups, BlasCtx c)
{
    const int rhs = blockIdx.x;
    if (!c.active[rhs]) return;
    double v = 0.0;
    const double* p = partial + (size_t)rhs * ngroups;
    // fixed order: thread k sums partials k, k + FIN_THREADS, ... (eight independent loads in flight), then the block tree
    int g = threadIdx.x;
    for (; g + 7 * FIN_THREADS < ngroups; g += 8 * FIN_THREADS) {
        double t[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) t[k] = p[g + k * FIN_THREADS];
#pragma unroll
        for (int k = 0; k < 8; ++k) v += t[k];
    }
    for (; g < ngroups; g += FIN_THREADS) v += p[g];
    const double tot = block_sum<FIN_THREADS>(v);
    if (threadIdx.x == 0) finish_scalar<FIN>(c, rhs, tot);
}

// iteration `iter` (0-based): x += alpha p for every rhs whose alpha belongs to this iteration (also the one that has just
// converged); p = r + beta p for the rhs that are still active.  The search direction is read from pin_ and written to p_ (the
// same stack from iteration 1 on; in iteration 0 pin_ is the right-hand side b itself, p_0 = r_0 = b, so no copies of b are made)
template <int PREC>
__global__ void __launch_bounds__(BLAS_THREADS) update_xp_kernel(int Vh, VecArg x_, VecArg p_, VecArg pin_, VecArg r_, BlasCtx c, int iter)
{
    typedef typename Prec<PREC>::real real;
    const int rhs = blockIdx.y;
    if (c.scal[rhs].alpha_iter != iter || c.scal[rhs].alpha == 0.0) {
        // iteration 0 also sets the initial guess x_0 = 0 (no memset, no read of x): a right-hand side that does not iterate (zero
        // source, breakdown in the first step) gets its zeros here
        if (iter == 0) {
            real z[24];
#pragma unroll
            for (int k = 0; k < 24; ++k) z[k] = 0;
            for (int cb = blockIdx.x * BLAS_THREADS + threadIdx.x; cb < Vh; cb += gridDim.x * BLAS_THREADS)
                store_spinor<PREC>(x_.p + rhs * x_.stride, Vh, cb, z);
        }
        return;
    }
    const bool more = c.active[rhs] != 0;
    const real alpha = (real)c.scal[rhs].alpha, beta = (real)c.scal[rhs].beta;
    for (int cb = blockIdx.x * BLAS_THREADS + threadIdx.x; cb < Vh; cb += gridDim.x * BLAS_THREADS) {
        real x[24], p[24];
        if (iter == 0) {
#pragma unroll
            for (int k = 0; k < 24; ++k) x[k] = 0;
        } else {
            load_spinor<PREC>(x_.p + rhs * x_.stride, Vh, cb, x);
        }
        load_spinor<PREC>(pin_.p + rhs * pin_.stride, Vh, cb, p);
#pragma unroll
        for (int k = 0; k < 24; ++k) x[k] = fma(alpha, p[k], x[k]);
        store_spinor<PREC>(x_.p + rhs * x_.stride, Vh, cb, x);
        if (more) {
            real r[24];
            load_spinor<PREC>(r_.p + rhs * r_.stride, Vh, cb, r);
#pragma unroll
            for (int k = 0; k < 24; ++k) p[k] = fma(beta, p[k], r[k]);
            store_spinor<PREC>(p_.p + rhs * p_.stride, Vh, cb, p);
        }
    }
}

// ---- search-direction ring of the truncated solver ------------------------------------------------------------------
// With room for LP_RING_DEPTH search directions the solution is not touched inside the iteration: iteration k only forms
// p_{k+1} = r_{k+1} + beta_k p_k into the next ring slot (three vector passes instead of five) and records alpha_k;
// x += sum_k alpha_k p_k is formed every LP_FLUSH_EVERY iterations and at the end in one pass over the kept directions (fp32 / fp64
// registers, one rounding to storage per pass).  Depth and schedule are constants, so a right-hand side gets the same bits whether
// it is solved alone or in a batch.
constexpr int LP_RING_DEPTH = 14;
constexpr int LP_FLUSH_EVERY = 12;

// p_out = r + beta p_in for the right-hand sides still active; hist[rhs] = alpha of iteration `iter` (0 if the rhs did not iterate)
template <int PREC>
__global__ void __launch_bounds__(BLAS_THREADS) update_p_hist_kernel(int Vh, VecArg pout_, VecArg pin_, VecArg r_, BlasCtx c, int iter,
                                                                     double* hist)
{
    typedef typename Prec<PREC>::real real;
    const int rhs = blockIdx.y;
    const double a = (c.scal[rhs].alpha_iter == iter) ? c.scal[rhs].alpha : 0.0;
    if (blockIdx.x == 0 && threadIdx.x == 0) hist[rhs] = a;
    if (a == 0.0 || c.active[rhs] == 0) return;
    const real beta = (real)c.scal[rhs].beta;
    for (int cb = blockIdx.x * BLAS_THREADS + threadIdx.x; cb < Vh; cb += gridDim.x * BLAS_THREADS) {
        real p[24], r[24];
        load_spinor<PREC>(pin_.p + rhs * pin_.stride, Vh, cb, p);
        load_spinor<PREC>(r_.p + rhs * r_.stride, Vh, cb, r);
#pragma unroll
        for (int k = 0; k < 24; ++k) p[k] = fma(beta, p[k], r[k]);
        store_spinor<PREC>(pout_.p + rhs * pout_.stride, Vh, cb, p);
    }
}

struct XTerms {
    const char* p[LP_FLUSH_EVERY];      // search directions (stacks over the right-hand sides)
    size_t stride[LP_FLUSH_EVERY];
    const double* alpha[LP_FLUSH_EVERY]; // their coefficients, [rhs]
    int n;
};

// x = (init ? 0 : x) + sum_{j < n} alpha_j p_j, terms in the order given, per right-hand side
template <int PREC>
__global__ void __launch_bounds__(BLAS_THREADS) accumulate_x_kernel(int Vh, VecArg x_, XTerms t, int init)
{
    typedef typename Prec<PREC>::real real;
    const int rhs = blockIdx.y;
    real a[LP_FLUSH_EVERY];
    bool any = false;
#pragma unroll
    for (int j = 0; j < LP_FLUSH_EVERY; ++j) {
        a[j] = j < t.n ? (real)t.alpha[j][rhs] : real(0);
        any |= a[j] != real(0);
    }
    if (!any && !init) return;
    for (int cb = blockIdx.x * BLAS_THREADS + threadIdx.x; cb < Vh; cb += gridDim.x * BLAS_THREADS) {
        real x[24];
        if (init) {
#pragma unroll
            for (int k = 0; k < 24; ++k) x[k] = 0;
        } else {
            load_spinor<PREC>(x_.p + rhs * x_.stride, Vh, cb, x);
        }
#pragma unroll
        for (int j = 0; j < LP_FLUSH_EVERY; ++j) {
            if (j < t.n && a[j] != real(0)) {
                real p[24];
                load_spinor<PREC>(t.p[j] + rhs * t.stride[j], Vh, cb, p);
#pragma unroll
                for (int k = 0; k < 24; ++k) x[k] = fma(a[j], p[k], x[k]);
            }
        }
        store_spinor<PREC>(x_.p + rhs * x_.stride, Vh, cb, x);
    }
}

static inline int blas_blocks(int Vh)
{
    int nb = (Vh + BLAS_THREADS - 1) / BLAS_THREADS;
    return nb > BLAS_MAX_BLOCKS ? BLAS_MAX_BLOCKS : nb;
}

} // namespace tmk
