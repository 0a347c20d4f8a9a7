// tm_dslash.cuh -- hopping term Dslash_{p <- pbar} with fused local epilogue.
//
//   (Dslash psi)(x) = sum_mu (1-g_mu) s U_mu(x) psi(x+mu) + (1+g_mu) s U_mu(x-mu)^dag psi(x-mu)
//   out = (p0 + i p1 g5) x + (q0 + i q1 g5) (Dslash in)                 (PAPER.md:384 fused kernels)
//
// One thread per output site and per group of NR right-hand sides.  Each link is loaded (and, for 12-real
// storage, rebuilt) once per thread and applied to NR half-spinors: spin projection happens before the colour
// multiply, so only 12 reals per neighbour go through the SU(3) product ((1 -+ g_mu) has rank 2).
// Threads of one CTA that share a site (threadIdx.y = rhs group) hit the same link lines in L1.
//
// Chiral basis, psi = (psi_0, psi_1 | psi_2, psi_3), e = +-1:
//   (1 - e g_1) psi: h0 = psi0 + e i psi3, h1 = psi1 + e i psi2; lower = (-e i h1, -e i h0)
//   (1 - e g_2) psi: h0 = psi0 + e   psi3, h1 = psi1 - e   psi2; lower = (-e   h1,  e   h0)
//   (1 - e g_3) psi: h0 = psi0 + e i psi2, h1 = psi1 - e i psi3; lower = (-e i h0,  e i h1)
//   (1 - e g_4) psi: h0 = psi0 - e   psi2, h1 = psi1 - e   psi3; lower = (-e   h0, -e   h1)
// e is a run-time +-1 (dagger flips it): every +- becomes one FMA, so the daggered operator costs nothing extra.
#pragma once
#include "tm_layout.cuh"

namespace tmk {

struct DslashKArgs {
    Geo g;
    const char* gauge;
    char* out;
    const char* in;
    const char* x;
    size_t link_block; // bytes of one (parity, mu) block
    size_t stride_out, stride_in, stride_x;
    const unsigned char* active;
    const char* link_cache; // optional: tile images built by link_cache_kernel (tm_dslash_tile.cuh)
    const char* dot_with;   // optional fused reduction: dot_partial[rhs][cb / 32] = sum over the warp of Re <dot_with, out>,
                            // or of |out|^2 if dot_with is null
    size_t stride_dot;
    double* dot_partial;
    // optional fused axpy: out = y - coef[rhs] * (epilogue result); coef is a device double per rhs (byte stride stride_coef)
    const char* axpy_y;
    size_t stride_y;
    const char* axpy_coef;
    size_t stride_coef;
    int parity; // of the output sites
    int nrhs;
    double eps;  // +1, or -1 for the daggered operator
    double pq[4];
};

// spin projection: h[12] = upper half of (1 - e g_mu) v
template <int MU, typename real>
__device__ __forceinline__ void spin_project(const real* v, real e, real* h)
{
    // v index: (s*3 + c)*2 + ri ; h index: (s*3 + c)*2 + ri, s = 0,1
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const real p0r = v[2 * c], p0i = v[2 * c + 1];
        const real p1r = v[6 + 2 * c], p1i = v[6 + 2 * c + 1];
        const real p2r = v[12 + 2 * c], p2i = v[12 + 2 * c + 1];
        const real p3r = v[18 + 2 * c], p3i = v[18 + 2 * c + 1];
        if (MU == 0) { // h0 = p0 + e i p3 ; h1 = p1 + e i p2
            h[2 * c] = fma(-e, p3i, p0r);
            h[2 * c + 1] = fma(e, p3r, p0i);
            h[6 + 2 * c] = fma(-e, p2i, p1r);
            h[6 + 2 * c + 1] = fma(e, p2r, p1i);
        } else if (MU == 1) { // h0 = p0 + e p3 ; h1 = p1 - e p2
            h[2 * c] = fma(e, p3r, p0r);
            h[2 * c + 1] = fma(e, p3i, p0i);
            h[6 + 2 * c] = fma(-e, p2r, p1r);
            h[6 + 2 * c + 1] = fma(-e, p2i, p1i);
        } else if (MU == 2) { // h0 = p0 + e i p2 ; h1 = p1 - e i p3
            h[2 * c] = fma(-e, p2i, p0r);
            h[2 * c + 1] = fma(e, p2r, p0i);
            h[6 + 2 * c] = fma(e, p3i, p1r);
            h[6 + 2 * c + 1] = fma(-e, p3r, p1i);
        } else { // h0 = p0 - e p2 ; h1 = p1 - e p3
            h[2 * c] = fma(-e, p2r, p0r);
            h[2 * c + 1] = fma(-e, p2i, p0i);
            h[6 + 2 * c] = fma(-e, p3r, p1r);
            h[6 + 2 * c + 1] = fma(-e, p3i, p1i);
        }
    }
}

// acc += (g, lower(g)) with the lower half rebuilt from the upper one
template <int MU, typename real>
__device__ __forceinline__ void spin_reconstruct(real* acc, const real* g, real e)
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const real g0r = g[2 * c], g0i = g[2 * c + 1], g1r = g[6 + 2 * c], g1i = g[6 + 2 * c + 1];
        acc[2 * c] += g0r;
        acc[2 * c + 1] += g0i;
        acc[6 + 2 * c] += g1r;
        acc[6 + 2 * c + 1] += g1i;
        if (MU == 0) { // lower = (-e i g1, -e i g0)
            acc[12 + 2 * c] = fma(e, g1i, acc[12 + 2 * c]);
            acc[12 + 2 * c + 1] = fma(-e, g1r, acc[12 + 2 * c + 1]);
            acc[18 + 2 * c] = fma(e, g0i, acc[18 + 2 * c]);
            acc[18 + 2 * c + 1] = fma(-e, g0r, acc[18 + 2 * c + 1]);
        } else if (MU == 1) { // lower = (-e g1, e g0)
            acc[12 + 2 * c] = fma(-e, g1r, acc[12 + 2 * c]);
            acc[12 + 2 * c + 1] = fma(-e, g1i, acc[12 + 2 * c + 1]);
            acc[18 + 2 * c] = fma(e, g0r, acc[18 + 2 * c]);
            acc[18 + 2 * c + 1] = fma(e, g0i, acc[18 + 2 * c + 1]);
        } else if (MU == 2) { // lower = (-e i g0, e i g1)
            acc[12 + 2 * c] = fma(e, g0i, acc[12 + 2 * c]);
            acc[12 + 2 * c + 1] = fma(-e, g0r, acc[12 + 2 * c + 1]);
            acc[18 + 2 * c] = fma(-e, g1i, acc[18 + 2 * c]);
            acc[18 + 2 * c + 1] = fma(e, g1r, acc[18 + 2 * c + 1]);
        } else { // lower = (-e g0, -e g1)
            acc[12 + 2 * c] = fma(-e, g0r, acc[12 + 2 * c]);
            acc[12 + 2 * c + 1] = fma(-e, g0i, acc[12 + 2 * c + 1]);
            acc[18 + 2 * c] = fma(-e, g1r, acc[18 + 2 * c]);
            acc[18 + 2 * c + 1] = fma(-e, g1i, acc[18 + 2 * c + 1]);
        }
    }
}

// g = U h (DAG = 0) or U^dag h (DAG = 1) for the two spin components of a half-spinor: 2 x 66 flops
template <int DAG, typename real>
__device__ __forceinline__ void su3_mul(const real* u, const real* h, real* g)
{
#pragma unroll
    for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            real re = 0, im = 0;
#pragma unroll
            for (int b = 0; b < 3; ++b) {
                const real ur = DAG ? u[2 * (b * 3 + a)] : u[2 * (a * 3 + b)];
                const real ui = DAG ? -u[2 * (b * 3 + a) + 1] : u[2 * (a * 3 + b) + 1];
                const real hr = h[6 * s + 2 * b], hi = h[6 * s + 2 * b + 1];
                re = fma(ur, hr, re);
                re = fma(-ui, hi, re);
                im = fma(ur, hi, im);
                im = fma(ui, hr, im);
            }
            g[6 * s + 2 * a] = re;
            g[6 * s + 2 * a + 1] = im;
        }
}

// out = y - coef[rhs] * o  (the CG residual update r -= alpha A p done in the epilogue that produces A p)
template <int PREC>
__device__ __forceinline__ void fused_axpy(const DslashKArgs& a, int rhs, int cb, typename Prec<PREC>::real* o)
{
    typedef typename Prec<PREC>::real real;
    real y[24];
    load_spinor<PREC, 2>(a.axpy_y + (size_t)rhs * a.stride_y, a.g.Vh, cb, y); // coherent: y may be the output vector (r -= alpha A p)
    const real c = (real)(*reinterpret_cast<const double*>(a.axpy_coef + (size_t)rhs * a.stride_coef));
#pragma unroll
    for (int k = 0; k < 24; ++k) o[k] = fma(-c, o[k], y[k]);
}

// Fused CG reduction: Re <w, out> (or |out|^2 when there is no w) of one site in the arithmetic precision, summed over the warp's 32
// consecutive sites in fp64 with a fixed shuffle tree; lane 0 stores the partial of site group cb / 32.  `o` is the
// epilogue result before storage rounding.  Every valid lane of the warp (cb < Vh) calls this.
template <int PREC>
__device__ __forceinline__ void warp_dot_store(const DslashKArgs& a, int rhs, int cb, const typename Prec<PREC>::real* o)
{
    typedef typename Prec<PREC>::real real;
    real s = 0;
    if (a.dot_with != nullptr) {
        real w[24];
        load_spinor<PREC>(a.dot_with + (size_t)rhs * a.stride_dot, a.g.Vh, cb, w);
#pragma unroll
        for (int k = 0; k < 24; ++k) s = fma(w[k], o[k], s);
    } else { // |out|^2
#pragma unroll
        for (int k = 0; k < 24; ++k) s = fma(o[k], o[k], s);
    }
    double v = (double)s;
    // The warp is 32 consecutive sites starting at a multiple of 32, so its valid lanes are [0, n) with n fixed by the geometry:
    // the mask does not depend on how the compiler reconverged the code above (an __activemask() taken after divergent code
    // could name fewer lanes and silently drop partial sums).
    const int lane = threadIdx.x & 31;
    const int n = min(32, a.g.Vh - (cb - lane));
    const unsigned m = n >= 32 ? 0xffffffffu : ((1u << n) - 1u);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        const double t = __shfl_down_sync(m, v, off);
        if (lane + off < n) v += t;
    }
    if (lane == 0) a.dot_partial[(size_t)rhs * ((a.g.Vh + 31) >> 5) + (cb >> 5)] = v;
}

template <int PREC, int RECON, int NR, int MU, int FWD>
__device__ __forceinline__ void hop_dir(const DslashKArgs& a, int cb, int nb, typename Prec<PREC>::real eps,
                                        typename Prec<PREC>::real sgn, const char* in0, const bool* act,
                                        typename Prec<PREC>::real (*acc)[24])
{
    typedef typename Prec<PREC>::real real;
    real u[18];
    const char* blk = a.gauge + (size_t)((FWD ? a.parity : 1 - a.parity) * 4 + MU) * a.link_block;
    load_link<PREC, RECON>(blk, a.g.Vh, FWD ? cb : nb, u);
    const real e = FWD ? eps : -eps;
#pragma unroll
    for (int r = 0; r < NR; ++r) {
        if (NR > 1 && !act[r]) continue;
        real v[24], h[12], g[12];
        load_spinor<PREC>(in0 + (size_t)r * a.stride_in, a.g.Vh, nb, v);
        spin_project<MU>(v, e, h);
        if (MU == 3) {
#pragma unroll
            for (int k = 0; k < 12; ++k) h[k] *= sgn;
        }
        su3_mul<FWD ? 0 : 1>(u, h, g);
        spin_reconstruct<MU>(acc[r], g, e);
    }
}

template <int PREC, int RECON, int NR>
__global__ void __launch_bounds__(256, PREC == 8 && NR == 1 ? 2 : 1) dslash_kernel(const DslashKArgs a)
{
    typedef typename Prec<PREC>::real real;
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= a.g.Vh) return;
    const int r0 = (blockIdx.y * blockDim.y + threadIdx.y) * NR;

    bool act[NR];
    bool any = false;
#pragma unroll
    for (int r = 0; r < NR; ++r) {
        act[r] = (a.active == nullptr) || (a.active[r0 + r] != 0);
        any |= act[r];
    }
    if (!any) return;

    // checkerboard coordinates (SURVEY.md 8(c-4) "Checkerboard neighbour indexing")
    uint32_t t, rem, z, rem2, y, xh;
    a.g.dXh.divmod((uint32_t)cb, rem, xh); // rem = cb / Xh (row index), xh = cb % Xh
    a.g.dY.divmod(rem, rem2, y);           // rem2 = row / Y, y = row % Y
    a.g.dZ.divmod(rem2, t, z);             // t = rem2 / Z, z = rem2 % Z
    const int xodd = (a.parity + y + z + t) & 1;
    const int Xh = a.g.Xh, XhY = a.g.XhY, V3h = a.g.V3h, Vh = a.g.Vh;
    const int nxp = cb + (xodd ? ((int)xh == Xh - 1 ? 1 - Xh : 1) : 0);
    const int nxm = cb - (xodd ? 0 : ((int)xh == 0 ? 1 - Xh : 1));
    const int nyp = cb + ((int)y == a.g.Y - 1 ? Xh - XhY : Xh);
    const int nym = cb - ((int)y == 0 ? Xh - XhY : Xh);
    const int nzp = cb + ((int)z == a.g.Z - 1 ? XhY - V3h : XhY);
    const int nzm = cb - ((int)z == 0 ? XhY - V3h : XhY);
    const int ntp = cb + ((int)t == a.g.T - 1 ? V3h - Vh : V3h);
    const int ntm = cb - ((int)t == 0 ? V3h - Vh : V3h);
    const real sgn_p = (a.g.ap && (int)t == a.g.T - 1) ? real(-1) : real(1);
    const real sgn_m = (a.g.ap && (int)t == 0) ? real(-1) : real(1);

    const real eps = (real)a.eps;
    const char* in0 = a.in + (size_t)r0 * a.stride_in;

    real acc[NR][24];
#pragma unroll
    for (int r = 0; r < NR; ++r)
#pragma unroll
        for (int k = 0; k < 24; ++k) acc[r][k] = 0;

    hop_dir<PREC, RECON, NR, 0, 1>(a, cb, nxp, eps, real(1), in0, act, acc);
    hop_dir<PREC, RECON, NR, 0, 0>(a, cb, nxm, eps, real(1), in0, act, acc);
    hop_dir<PREC, RECON, NR, 1, 1>(a, cb, nyp, eps, real(1), in0, act, acc);
    hop_dir<PREC, RECON, NR, 1, 0>(a, cb, nym, eps, real(1), in0, act, acc);
    hop_dir<PREC, RECON, NR, 2, 1>(a, cb, nzp, eps, real(1), in0, act, acc);
    hop_dir<PREC, RECON, NR, 2, 0>(a, cb, nzm, eps, real(1), in0, act, acc);
    hop_dir<PREC, RECON, NR, 3, 1>(a, cb, ntp, eps, sgn_p, in0, act, acc);
    hop_dir<PREC, RECON, NR, 3, 0>(a, cb, ntm, eps, sgn_m, in0, act, acc);

    // epilogue: out = (p0 + i p1 g5) x + (q0 + i q1 g5) acc ; g5 = diag(1,1,-1,-1)
    const real p0 = (real)a.pq[0], p1 = (real)a.pq[1], q0 = (real)a.pq[2], q1 = (real)a.pq[3];
#pragma unroll
    for (int r = 0; r < NR; ++r) {
        if (NR > 1 && !act[r]) continue;
        real o[24];
#pragma unroll
        for (int k = 0; k < 12; ++k) {
            const real s5 = (k < 6) ? real(1) : real(-1);
            const real dr = acc[r][2 * k], di = acc[r][2 * k + 1];
            o[2 * k] = q0 * dr - s5 * q1 * di;
            o[2 * k + 1] = q0 * di + s5 * q1 * dr;
        }
        if (a.x != nullptr) {
            real xv[24];
            load_spinor<PREC, 1>(a.x + (size_t)(r0 + r) * a.stride_x, Vh, cb, xv);
#pragma unroll
            for (int k = 0; k < 12; ++k) {
                const real s5 = (k < 6) ? real(1) : real(-1);
                o[2 * k] += p0 * xv[2 * k] - s5 * p1 * xv[2 * k + 1];
                o[2 * k + 1] += p0 * xv[2 * k + 1] + s5 * p1 * xv[2 * k];
            }
        }
        if (a.axpy_y != nullptr) fused_axpy<PREC>(a, r0 + r, cb, o);
        store_spinor<PREC>(a.out + (size_t)(r0 + r) * a.stride_out, Vh, cb, o);
        if (a.dot_partial != nullptr) warp_dot_store<PREC>(a, r0 + r, cb, o);
    }
}

// host-side launcher for one (PREC, RECON); defined per translation unit via TM_INSTANTIATE_DSLASH
template <int PREC, int RECON>
int launch_dslash_t(const Geo& g, const DslashParams& p, cudaStream_t st);

template <int PREC, int RECON, int NR>
static inline void launch_nr(const DslashKArgs& a, int groups, cudaStream_t st)
{
    int gy = 1;
    for (int d = 4; d >= 1; --d)
        if (groups % d == 0) { gy = d; break; }
    const int bx = (gy == 1) ? 128 : 64;
    dim3 block(bx, gy), grid((a.g.Vh + bx - 1) / bx, groups / gy);
    dslash_kernel<PREC, RECON, NR><<<grid, block, 0, st>>>(a);
}

} // namespace tmk
