// tm_insert.cu -- SURVEY.md 8(f) NEXT-2 / NEXT-3: what the paper's contraction kernels and variance-reduction drivers add
// to the hot path (PAPER.md:407-415 App. A.2 "Contraction kernels", :148-169 time-dilution and HPE, :421-427 FFT + p^2 cut).
//
//   tm_covdev            (D_mu psi)(x) = 1/2 [s U_mu(x) psi(x+mu) - s U_mu(x-mu)^dag psi(x-mu)]   "covariant-derivative kernel"
//   tm_contract_field    C[x][al][be] = sum_c conj(a_{al c}(x)) b_{be c}(x)                        colour traced, Dirac + volume open
//   tm_loop_momentum     L[n][t][k] = sum_xvec exp(-i p_k xvec) a^dag Gamma_n b                     contraction fused with a separable
//                        partial DFT (x, then y, then z) for the few momenta kept (p^2 <= 9), instead of the paper's
//                        field -> cuFFT -> cut: the 256 B/site field never goes to HBM
//   tm_time_dilute       noise restricted to chosen time slices (time dilution, coherent sources)
//   tm_hpe_remainder     (B H)^4 s, B = R^-1, H = -kappa Dslash: the stochastic term of Eq. (17)
//   tm_hpe_local_traces  per-site Tr[Gamma_n (B - BHB + (BH)^2 B - (BH)^3 B)]_xx, the exact terms of Eq. (16) for ultra-local X
// (tm_loop_contract_slice, the single-time-slice contraction, lives in tm_loop.cu.)
#include <cmath>
#include <cstring>
#include "tm_dslash_tile.cuh"
#include "tm_gamma.cuh"
#include "tm_contract.cuh"

namespace tmk {

// ---- covariant derivative ----------------------------------------------------------------------------------------
// One thread per site of one parity; spin is untouched, so the two SU(3) products act on all four spin components.
template <int PREC, int RECON>
__global__ void __launch_bounds__(128) covdev_kernel(Geo g, const char* gauge, size_t link_block, char* out_full, const char* in_full,
                                                     size_t parity_bytes, int mu)
{
    typedef typename Prec<PREC>::real real;
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    const int parity = blockIdx.y, rhs = blockIdx.z;
    if (cb >= g.Vh) return;
    int nb[8];
    float sgp, sgm;
    tile_neighbours(g, parity, cb, nb, sgp, sgm);
    const int nf = nb[2 * mu], nbk = nb[2 * mu + 1];
    const real sf = (mu == 3) ? (real)sgp : real(1), sb = (mu == 3) ? (real)sgm : real(1);
    const char* in = in_full + (size_t)rhs * 2 * parity_bytes + (size_t)(1 - parity) * parity_bytes;
    real u[18], v[24], gf[24], gb[24];
    load_link<PREC, RECON>(gauge + (size_t)(parity * 4 + mu) * link_block, g.Vh, cb, u);
    load_spinor<PREC>(in, g.Vh, nf, v);
    su3_mul<0>(u, v, gf);
    su3_mul<0>(u, v + 12, gf + 12);
    load_link<PREC, RECON>(gauge + (size_t)((1 - parity) * 4 + mu) * link_block, g.Vh, nbk, u);
    load_spinor<PREC>(in, g.Vh, nbk, v);
    su3_mul<1>(u, v, gb);
    su3_mul<1>(u, v + 12, gb + 12);
    real o[24];
    const real hf = real(0.5) * sf, hb = real(0.5) * sb;
#pragma unroll
    for (int k = 0; k < 24; ++k) o[k] = hf * gf[k] - hb * gb[k];
    store_spinor<PREC>(out_full + (size_t)rhs * 2 * parity_bytes + (size_t)parity * parity_bytes, g.Vh, cb, o);
}

template <int PREC, int RECON>
static int covdev_launch(const Geo& g, const void* gauge, void* out_full, const void* in_full, int mu, int nrhs, cudaStream_t st)
{
    dim3 grid((g.Vh + 127) / 128, 2, nrhs);
    covdev_kernel<PREC, RECON><<<grid, 128, 0, st>>>(g, (const char*)gauge, link_block_bytes(g, PREC, RECON), (char*)out_full,
                                                     (const char*)in_full, spinor_parity_bytes(g, PREC), mu);
    TM_LAUNCH_CHECK("covdev_kernel");
    return TM_OK;
}

// ---- contraction field -------------------------------------------------------------------------------------------
// C_{al be}(x) of one site in the storage arithmetic (fp32 for fp32 / fp16 fields), as in loop_partial_kernel
template <typename real>
__device__ __forceinline__ void site_contract(const real* a, const real* b, real* c32)
{
#pragma unroll
    for (int al = 0; al < 4; ++al)
#pragma unroll
        for (int be = 0; be < 4; ++be) {
            real re = 0, im = 0;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const real ar = a[(al * 3 + c) * 2], ai = a[(al * 3 + c) * 2 + 1];
                const real br = b[(be * 3 + c) * 2], bi = b[(be * 3 + c) * 2 + 1];
                re = fma(ar, br, re);
                re = fma(ai, bi, re);
                im = fma(ar, bi, im);
                im = fma(-ai, br, im);
            }
            c32[(al * 4 + be) * 2] = re;
            c32[(al * 4 + be) * 2 + 1] = im;
        }
}

// out[rhs][site][4][4][2] fp64, site lexicographic (x fastest) = 2 cb + (x odd): "fits exactly in the input required" by an
// FFT.  Each warp transposes its 32 x 32 doubles through shared memory so that the stores are coalesced.
template <int PREC>
__global__ void __launch_bounds__(128) contract_field_kernel(Geo g, const char* a_full, const char* b_full, size_t parity_bytes,
                                                             double* out, long long V)
{
    typedef typename Prec<PREC>::real real;
    __shared__ double tile[4][32][33];
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    const int parity = blockIdx.y, rhs = blockIdx.z;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const bool valid = cb < g.Vh;
    if (valid) {
        real a[24], b[24], c[32];
        load_spinor<PREC>(a_full + (size_t)rhs * 2 * parity_bytes + (size_t)parity * parity_bytes, g.Vh, cb, a);
        load_spinor<PREC>(b_full + (size_t)rhs * 2 * parity_bytes + (size_t)parity * parity_bytes, g.Vh, cb, b);
        site_contract<real>(a, b, c);
#pragma unroll
        for (int k = 0; k < 32; ++k) tile[warp][lane][k] = (double)c[k];
    }
    __syncwarp();
    const int cb0 = cb - lane;
    for (int s = 0; s < 32; ++s) {
        const int c2 = cb0 + s;
        if (c2 >= g.Vh) break;
        uint32_t row, xh, rem2, y, t, z;
        g.dXh.divmod((uint32_t)c2, row, xh);
        g.dY.divmod(row, rem2, y);
        g.dZ.divmod(rem2, t, z);
        const size_t site = 2 * (size_t)c2 + ((parity + y + z + t) & 1);
        out[((size_t)rhs * V + site) * 32 + lane] = tile[warp][s][lane];
    }
}

} // namespace tmk

namespace tmk {

// ---- momentum-projected loops --------------------------------------------------------------------------------------
// Stage 1 (one CTA per (z, t) plane and rhs): contraction of every site of the plane, DFT over x for the NP = 2 P + 1
// values n_x = -P..P, then over y, accumulated per thread in fp64 in a fixed order:
//     W2[rhs][t][z][ipx][ipy][ab] = sum_y e^{-2 pi i n_y y / Y} sum_x e^{-2 pi i n_x x / X} C_ab(x, y, z, t).
// Stage 2 (loop_mom_final_kernel): DFT over z for the listed momenta and the 16 Gamma_n.
constexpr int MOM_THREADS = 256;
constexpr int MOM_ROWS = 8;   // y rows contracted per pass (at most; MOM_THREADS / X when X > 32)
constexpr int MOM_MAXP = 4;   // |n_i| <= 4 (p^2 <= 9 needs 3)

__device__ __forceinline__ double2 cfma(double2 a, double2 b, double2 c)
{
    return make_double2(fma(a.x, b.x, fma(-a.y, b.y, c.x)), fma(a.x, b.y, fma(a.y, b.x, c.y)));
}
// exp(-2 pi i n k / N) with the argument reduced in integers first
__device__ __forceinline__ double2 dft_phase(int n, int k, int N)
{
    int m = (n * k) % N;
    if (m < 0) m += N;
    double s, c;
    sincospi(-2.0 * (double)m / (double)N, &s, &c);
    return make_double2(c, s);
}
// (cos, sin)(2 pi n k / N)
__device__ __forceinline__ double2 cos_sin(int n, int k, int N)
{
    double s, c;
    sincospi(2.0 * (double)((n * k) % N) / (double)N, &s, &c);
    return make_double2(c, s);
}

template <int PREC> struct MomC { typedef float2 type; };
template <> struct MomC<8> { typedef double2 type; };

// e^{-i n theta} = cos(n theta) - i sin(n theta): the sums over x (and y) are kept as real-weighted sums
//   Sc[n] = sum C cos(n theta), Ss[n] = sum C sin(n theta), n = 0..P, and +-n are combined at the end (half the multiplies
// of a complex DFT).  Every thread keeps its 2 P + 1 complex sums in registers and reads each C once.
template <int PREC, int P>
__global__ void __launch_bounds__(MOM_THREADS, PREC == 8 ? 2 : 3) loop_mom_plane_kernel(Geo g, const char* a_full, const char* b_full,
                                                                     size_t parity_bytes, int R, double2* W2)
{
    typedef typename Prec<PREC>::real real;
    typedef typename MomC<PREC>::type CT;
    extern __shared__ double2 smem[];
    constexpr int NP = 2 * P + 1;
    const int X = g.X, Y = g.Y;
    // x sums run in the storage arithmetic (fp32 for fp32 / fp16 fields: at most X terms per sum, like the LOOP_CHUNK sites of
    // loop_partial_kernel), everything after them in fp64
    typedef typename Prec<PREC>::real acc_t;
    double2* csy = smem;                          // [P+1][Y]  (cos, sin)(2 pi n y / Y)
    double2* Part = csy + (P + 1) * Y;            // [nseg][R][16][NP]
    const int nseg = max(1, MOM_THREADS / (R * 16));
    const int nh = min(4, MOM_THREADS / (NP * 16)); // row shares of step (3); Part also serves as their [nh][NP*16][NP] scratch
    CT* csx = reinterpret_cast<CT*>(Part + (size_t)max(nseg * R, nh * NP) * 16 * NP); // [P+1][X]
    CT* Cs = csx + (P + 1) * X;                   // [R][X][16]
    const int z = blockIdx.x, t = blockIdx.y, rhs = blockIdx.z, tid = threadIdx.x;
    for (int i = tid; i < (P + 1) * X; i += MOM_THREADS) {
        const double2 w = cos_sin(i / X, i % X, X);
        CT v;
        v.x = (acc_t)w.x;
        v.y = (acc_t)w.y;
        csx[i] = v;
    }
    for (int i = tid; i < (P + 1) * Y; i += MOM_THREADS) csy[i] = cos_sin(i / Y, i % Y, Y);
    double2 yc[P + 1], ys[P + 1];
#pragma unroll
    for (int m = 0; m <= P; ++m) yc[m] = ys[m] = make_double2(0.0, 0.0);
    const char* af = a_full + (size_t)rhs * 2 * parity_bytes;
    const char* bf = b_full + (size_t)rhs * 2 * parity_bytes;
    const int xseg = (X + nseg - 1) / nseg;
    __syncthreads();
    for (int y0 = 0; y0 < Y; y0 += R) {
        const int nr = min(R, Y - y0);
        // (1) contraction of the sites of rows y0 .. y0 + nr - 1, products in the storage arithmetic
        for (int i = tid; i < nr * X; i += MOM_THREADS) {
            const int r = i / X, x = i - r * X, y = y0 + r;
            const int parity = (x + y + z + t) & 1;
            const int cb = (x >> 1) + g.Xh * (y + Y * (z + g.Z * t));
            real a[24], b[24], c[32];
            load_spinor<PREC>(af + (size_t)parity * parity_bytes, g.Vh, cb, a);
            load_spinor<PREC>(bf + (size_t)parity * parity_bytes, g.Vh, cb, b);
            site_contract<real>(a, b, c);
#pragma unroll
            for (int k = 0; k < 16; ++k) {
                CT v;
                v.x = c[2 * k];
                v.y = c[2 * k + 1];
                Cs[(r * X + x) * 16 + k] = v;
            }
        }
        __syncthreads();
        // (2) sums over x: thread = (segment of x, row, ab)
        if (tid < nseg * R * 16) {
            const int ab = tid & 15, r = (tid >> 4) % R, seg = (tid >> 4) / R;
            if (r < nr) {
                acc_t scx[P + 1], scy[P + 1], ssx[P + 1], ssy[P + 1];
#pragma unroll
                for (int n = 0; n <= P; ++n) scx[n] = scy[n] = ssx[n] = ssy[n] = 0;
                const int x1 = min(X, (seg + 1) * xseg);
#pragma unroll 4
                for (int x = seg * xseg; x < x1; ++x) {
                    const CT cv = Cs[(r * X + x) * 16 + ab];
#pragma unroll
                    for (int n = 0; n <= P; ++n) {
                        const CT w = csx[n * X + x];
                        scx[n] = fma(cv.x, w.x, scx[n]);
                        scy[n] = fma(cv.y, w.x, scy[n]);
                        if (n > 0) {
                            ssx[n] = fma(cv.x, w.y, ssx[n]);
                            ssy[n] = fma(cv.y, w.y, ssy[n]);
                        }
                    }
                }
                double2* dst = Part + (size_t)((seg * R + r) * 16 + ab) * NP;
#pragma unroll
                for (int n = 0; n <= P; ++n)
                    if (n <= P) {
                        dst[n] = make_double2((double)scx[n], (double)scy[n]);
                        if (n > 0) dst[P + n] = make_double2((double)ssx[n], (double)ssy[n]);
                    }
            }
        }
        __syncthreads();
        // (3) sums over y: thread = (share of the rows, ipx, ab); W1 = sum_seg [Sc[|n|] - sgn(n) i Ss[|n|]].  No barrier after
        // this step: the next pass's contraction only writes Cs, and Part is rewritten after the next barrier.
        if (tid < nh * NP * 16) {
            const int item = tid % (NP * 16), half = tid / (NP * 16);
            const int ab = item & 15, n = (item >> 4) - P, an = n < 0 ? -n : n;
            const double sg = n > 0 ? 1.0 : (n < 0 ? -1.0 : 0.0);
            for (int r = half; r < nr; r += nh) {
                double2 w = make_double2(0.0, 0.0);
                for (int seg = 0; seg < nseg; ++seg) {
                    const double2* src = Part + (size_t)((seg * R + r) * 16 + ab) * NP;
                    const double2 c = src[an];
                    w.x += c.x;
                    w.y += c.y;
                    if (an > 0) {
                        const double2 sn = src[P + an];
                        w.x += sg * sn.y; // -i sg (sx + i sy) = sg sy - i sg sx
                        w.y -= sg * sn.x;
                    }
                }
#pragma unroll
                for (int m = 0; m <= P; ++m) {
                    const double2 q = csy[m * Y + y0 + r];
                    yc[m].x = fma(w.x, q.x, yc[m].x);
                    yc[m].y = fma(w.y, q.x, yc[m].y);
                    if (m > 0) {
                        ys[m].x = fma(w.x, q.y, ys[m].x);
                        ys[m].y = fma(w.y, q.y, ys[m].y);
                    }
                }
            }
        }
    }
    // combine the row shares in a fixed order (Part is free again after this barrier)
    __syncthreads();
    if (tid < nh * NP * 16) {
        double2* dst = Part + (size_t)tid * NP;
#pragma unroll
        for (int m = 0; m <= P; ++m) {
            dst[m] = yc[m];
            if (m > 0) dst[P + m] = ys[m];
        }
    }
    __syncthreads();
    if (tid < NP * 16) {
        for (int h = 1; h < nh; ++h) {
            const double2* src = Part + (size_t)(h * NP * 16 + tid) * NP;
#pragma unroll
            for (int m = 0; m <= P; ++m) {
                yc[m].x += src[m].x;
                yc[m].y += src[m].y;
                if (m > 0) {
                    ys[m].x += src[P + m].x;
                    ys[m].y += src[P + m].y;
                }
            }
        }
        const int ab = tid & 15, ipx = tid >> 4;
        double2* dst = W2 + (((size_t)rhs * g.T + t) * g.Z + z) * (NP * NP * 16);
#pragma unroll
        for (int m = 0; m <= P; ++m) {
            // n_y = +m: Yc - i Ys ; n_y = -m: Yc + i Ys
            dst[(ipx * NP + (P + m)) * 16 + ab] = make_double2(yc[m].x + ys[m].y, yc[m].y - ys[m].x);
            if (m > 0) dst[(ipx * NP + (P - m)) * 16 + ab] = make_double2(yc[m].x - ys[m].y, yc[m].y + ys[m].x);
        }
    }
}

// ---- stage 1 for fp32 / fp16 fields, X <= 64, Y <= 128: one warp per row, no CTA barrier inside the plane ----------------------
// CTA = one (z, t) plane of one right-hand side, warp w = the rows y in [8 w, 8 w + 8).  Per row:
//   (1) lane = site x: colour-traced contraction C[32 reals] (fp16 fields: exact products of the stored words, FHFMA) into a
//       warp-private shared-memory tile [x][33];
//   (2) lane = one of the 32 reals k = (ab, re/im): sums over x with REAL weights, even / odd split in x -> X - x (cos is even,
//       sin is odd: half the multiplies): Sc[n] = sum C cos(n th x), Ss[n] = sum C sin(n th x), n <= P; the weights are warp
//       uniform and come from the kernel parameters (constant bank), not from shared memory;
//   (3) sums over y into (2P+1)^2 fp32 registers per lane (at most 8 rows, the LOOP_CHUNK rule of the loop kernel).
// The warps' partials are then added in fp64 in a fixed order and turned into W2[ipx][ipy][ab] (the layout stage 2 reads).
struct MomWeights {
    float xc[MOM_MAXP + 1][32];            // cos(2 pi n j / X), j < X/2
    float xs[MOM_MAXP + 1][32];            // sin(2 pi n j / X)
    float yw[128][2 * MOM_MAXP + 1];       // row y: cos(2 pi m y / Y), m = 0..P, then sin(2 pi m y / Y), m = 1..P
};
constexpr int MOMR_ROWS = 8; // rows per warp
// CTAs per SM asked of the compiler for the 4-warp shape (B200 sweep at 32^3 x 64, 12 sources, 123 momenta): fp16 storage 1122 / 1022 /
// 986 / 1082 us at 4 / 5 / 6 / 8, fp32 1163 / 1215 / 1213 / 1587 us
template <int PREC> struct MomrMinb { static constexpr int value = PREC == 2 ? 6 : 4; };

// XH: X / 2 as a compile-time constant (the x loop is unrolled: tile reads and weights become immediates), 0 = run-time X.
// MAXT / MINB: launch bounds (threads per CTA = 32 x ceil(Y / 8)).
template <int PREC, int P, int XH, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) loop_mom_row_kernel(Geo g, const char* a_full, const char* b_full, size_t parity_bytes,
                                                                  const __grid_constant__ MomWeights W, double2* W2)
{
    constexpr int NX = 2 * P + 1;
    extern __shared__ float msm[];
    const int X = XH ? 2 * XH : g.X, Y = g.Y, XT = X > 32 ? 64 : 32;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    float* tile = msm + (size_t)warp * XT * 33; // [x][33]
    float* part = msm + (size_t)warp * NX * NX * 32; // [xi][yi][k]; written after every warp is done with its tile
    const int z = blockIdx.x, t = blockIdx.y, rhs = blockIdx.z;
    const char* af = a_full + (size_t)rhs * 2 * parity_bytes;
    const char* bf = b_full + (size_t)rhs * 2 * parity_bytes;
    float acc[NX][NX];
#pragma unroll
    for (int i = 0; i < NX; ++i)
#pragma unroll
        for (int j = 0; j < NX; ++j) acc[i][j] = 0.f;
    const int y1 = min(Y, (warp + 1) * MOMR_ROWS);
    for (int y = warp * MOMR_ROWS; y < y1; ++y) {
        // (1) contraction of the row
        for (int x = lane; x < X; x += 32) {
            const int parity = (x + y + z + t) & 1;
            const int cb = (x >> 1) + g.Xh * (y + Y * (z + g.Z * t));
            float c[32];
            if constexpr (PREC == 2) {
                uint4 qa[3], qb[3];
                const uint4* pa = reinterpret_cast<const uint4*>(af + (size_t)parity * parity_bytes) + cb;
                const uint4* pb = reinterpret_cast<const uint4*>(bf + (size_t)parity * parity_bytes) + cb;
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    qa[k] = __ldg(pa + (size_t)k * g.Vh);
                    qb[k] = __ldg(pb + (size_t)k * g.Vh);
                }
                const float na = __ldg(reinterpret_cast<const float*>(reinterpret_cast<const uint4*>(af + (size_t)parity * parity_bytes) + (size_t)3 * g.Vh) + cb);
                const float nb_ = __ldg(reinterpret_cast<const float*>(reinterpret_cast<const uint4*>(bf + (size_t)parity * parity_bytes) + (size_t)3 * g.Vh) + cb);
#pragma unroll
                for (int k = 0; k < 32; ++k) c[k] = 0.f;
                site_contract_h(qa, na, qb, nb_, c);
            } else {
                float a[24], b[24];
                load_spinor<PREC>(af + (size_t)parity * parity_bytes, g.Vh, cb, a);
                load_spinor<PREC>(bf + (size_t)parity * parity_bytes, g.Vh, cb, b);
                site_contract<float>(a, b, c);
            }
#pragma unroll
            for (int k = 0; k < 32; ++k) tile[x * 33 + k] = c[k];
        }
        __syncwarp();
        // (2) sums over x for the real k = lane
        float S[NX];
        {
            const float e0 = tile[lane], eh = tile[(X >> 1) * 33 + lane];
#pragma unroll
            for (int n = 0; n <= P; ++n) S[n] = (n & 1) ? e0 - eh : e0 + eh;
#pragma unroll
            for (int n = 1; n <= P; ++n) S[P + n] = 0.f;
#pragma unroll
            for (int j = 1; j < (XH ? XH : (X >> 1)); ++j) {
                const float cj = tile[j * 33 + lane], cm = tile[(X - j) * 33 + lane];
                const float e = cj + cm, o = cj - cm;
                S[0] += e;
#pragma unroll
                for (int n = 1; n <= P; ++n) {
                    S[n] = fmaf(e, W.xc[n][j], S[n]);
                    S[P + n] = fmaf(o, W.xs[n][j], S[P + n]);
                }
            }
        }
        __syncwarp(); // the tile is free for the next row
        // (3) sums over y
#pragma unroll
        for (int yi = 0; yi < NX; ++yi) {
            const float wy = yi == 0 ? 1.f : W.yw[y][yi];
#pragma unroll
            for (int xi = 0; xi < NX; ++xi) acc[xi][yi] = yi == 0 ? acc[xi][yi] + S[xi] : fmaf(S[xi], wy, acc[xi][yi]);
        }
    }
    __syncthreads(); // the partials alias the tiles
#pragma unroll
    for (int xi = 0; xi < NX; ++xi)
#pragma unroll
        for (int yi = 0; yi < NX; ++yi) part[(xi * NX + yi) * 32 + lane] = acc[xi][yi];
    __syncthreads();
    // combine: item = (ipx, ipy, ab); A(xi, yi, k) = sum over the warps in fp64, fixed order
    const float* part0 = msm;
    double2* dst = W2 + (((size_t)rhs * g.T + t) * g.Z + z) * (NX * NX * 16);
    for (int item = threadIdx.x; item < NX * NX * 16; item += blockDim.x) {
        const int ab = item & 15, ipy = (item >> 4) % NX, ipx = (item >> 4) / NX;
        const int nx = ipx - P, ny = ipy - P, ax = nx < 0 ? -nx : nx, ay = ny < 0 ? -ny : ny;
        const double sx = nx > 0 ? 1.0 : (nx < 0 ? -1.0 : 0.0), sy = ny > 0 ? 1.0 : (ny < 0 ? -1.0 : 0.0);
        double v[4][2]; // (cc, cs, sc, ss) x (re, im)
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int xi = (q & 2) ? P + ax : ax, yi = (q & 1) ? P + ay : ay;
            const bool on = !((q & 2) && ax == 0) && !((q & 1) && ay == 0);
#pragma unroll
            for (int ri = 0; ri < 2; ++ri) {
                double sum = 0.0;
                if (on)
                    for (int w = 0; w < nwarp; ++w) sum += (double)part0[((size_t)w * NX * NX + (xi * NX + yi)) * 32 + 2 * ab + ri];
                v[q][ri] = sum;
            }
        }
        // sum C (cos_x - i sx sin_x)(cos_y - i sy sin_y), C = Cr + i Ci
        const double re = v[0][0] - sx * sy * v[3][0] + (sy * v[1][1] + sx * v[2][1]);
        const double im = v[0][1] - sx * sy * v[3][1] - (sy * v[1][0] + sx * v[2][0]);
        dst[(ipx * NX + ipy) * 16 + ab] = make_double2(re, im);
    }
}

// out[rhs][n][t][k] = sum_ab (Gamma_n)_ab sum_z e^{-2 pi i n_z z / Z} W2[rhs][t][z][ipx_k][ipy_k][ab]; 8 momenta per CTA
__global__ void __launch_bounds__(128) loop_mom_final_kernel(Geo g, int P, const double2* W2, const int* mom, int K, GammaTable tb,
                                                             double* out)
{
    __shared__ double2 Ck[8][16];
    __shared__ double2 ph[256]; // e^{-2 pi i m / Z}, m < Z (Z <= 256; larger Z evaluates the phase per term)
    const int t = blockIdx.x, rhs = blockIdx.y;
    const int NP = 2 * P + 1, nout = NP * NP * 16;
    const int kk = threadIdx.x >> 4, ab = threadIdx.x & 15;
    const int k = blockIdx.z * 8 + kk;
    const bool table = g.Z <= 256;
    if (table)
        for (int m = threadIdx.x; m < g.Z; m += blockDim.x) ph[m] = dft_phase(1, m, g.Z);
    __syncthreads();
    if (k < K) {
        const int nx = mom[3 * k], ny = mom[3 * k + 1], nz = mom[3 * k + 2];
        const double2* src = W2 + ((size_t)rhs * g.T + t) * g.Z * nout + ((nx + P) * NP + (ny + P)) * 16 + ab;
        double2 s = make_double2(0.0, 0.0);
        int m = 0;                                   // (nz z) mod Z, stepped
        const int step = ((nz % g.Z) + g.Z) % g.Z;
        for (int z = 0; z < g.Z; ++z) {
            s = cfma(src[(size_t)z * nout], table ? ph[m] : dft_phase(nz, z, g.Z), s);
            m += step;
            if (m >= g.Z) m -= g.Z;
        }
        Ck[kk][ab] = s;
    }
    __syncthreads();
    if (k < K) {
        const int n = ab;
        double re = 0.0, im = 0.0;
#pragma unroll
        for (int al = 0; al < 4; ++al) {
            const int be = tb.col[n][al];
            const double gr = tb.re[n][al], gi = tb.im[n][al];
            const double2 c = Ck[kk][al * 4 + be];
            re += gr * c.x - gi * c.y;
            im += gr * c.y + gi * c.x;
        }
        double* o = out + ((((size_t)rhs * 16 + n) * g.T + t) * K + k) * 2;
        o[0] = re;
        o[1] = im;
    }
}

static size_t mom_w2_bytes(const Geo& g, int P, int nrhs)
{
    const size_t NP = 2 * P + 1;
    return round256((size_t)nrhs * g.T * g.Z * NP * NP * 16 * sizeof(double2));
}
static int mom_rows(const Geo& g)
{
    int R = MOM_THREADS / g.X;
    if (R > MOM_ROWS) R = MOM_ROWS;
    if (R < 1) R = 1;
    if (R > g.Y) R = g.Y;
    return R;
}
static size_t mom_smem_bytes(const Geo& g, int P, int prec)
{
    const size_t NP = 2 * P + 1, R = mom_rows(g);
    const size_t nseg = MOM_THREADS / (R * 16) > 0 ? MOM_THREADS / (R * 16) : 1;
    size_t nh = MOM_THREADS / (NP * 16);
    if (nh > 4) nh = 4;
    const size_t part = (nseg * R > nh * NP ? nseg * R : nh * NP) * 16 * NP;
    return ((size_t)(P + 1) * g.Y + part) * sizeof(double2) + ((size_t)(P + 1) * g.X + R * g.X * 16) * (prec == 8 ? sizeof(double2) : sizeof(float2));
}

} // namespace tmk

namespace tmk {

// ---- time dilution -------------------------------------------------------------------------------------------------
struct TimeMask {
    unsigned int bits[16]; // T <= 512
};

// packed full-lattice spinors are arrays [rhs][parity][chunk][cb] of 16-byte chunks (+ fp32 norms for fp16) and a time
// slice is the contiguous cb range [t V3h, (t+1) V3h): element-wise copy-or-zero.
__global__ void time_dilute_kernel(Geo g, const char* in, char* out, size_t parity_bytes, int nchunk, int has_norm, TimeMask m)
{
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= g.Vh) return;
    const size_t base = (size_t)blockIdx.y * parity_bytes; // blockIdx.y = rhs * 2 + parity
    const int t = cb / g.V3h;
    const bool keep = (m.bits[t >> 5] >> (t & 31)) & 1u;
    const uint4* src = reinterpret_cast<const uint4*>(in + base);
    uint4* dst = reinterpret_cast<uint4*>(out + base);
    for (int k = 0; k < nchunk; ++k) dst[(size_t)k * g.Vh + cb] = keep ? src[(size_t)k * g.Vh + cb] : make_uint4(0, 0, 0, 0);
    if (has_norm) {
        const float* sn = reinterpret_cast<const float*>(src + (size_t)nchunk * g.Vh);
        float* dn = reinterpret_cast<float*>(dst + (size_t)nchunk * g.Vh);
        dn[cb] = keep ? sn[cb] : 0.f;
    }
}

// ---- hopping-parameter expansion --------------------------------------------------------------------------------------
// out_full = (B H) in_full on both parities: B H = -kappa R^-1 Dslash, R^-1 = (1 - i a g5) / (1 + a^2), a = 2 kappa mu
static int hpe_BH(const Geo& g, const void* gauge, int prec, int recon, void* out_full, const void* in_full, double kappa, double mu,
                  int nrhs, cudaStream_t st)
{
    const size_t pb = spinor_parity_bytes(g, prec);
    const double a = 2.0 * kappa * mu, d = 1.0 / (1.0 + a * a);
    DslashParams p;
    p.gauge = gauge; p.nrhs = nrhs; p.active = nullptr; p.dagger = 0; p.x = nullptr;
    p.rhs_stride_out = p.rhs_stride_in = p.rhs_stride_x = 2 * pb;
    p.pq[0] = 0.0; p.pq[1] = 0.0; p.pq[2] = -kappa * d; p.pq[3] = kappa * a * d;
    for (int parity = 0; parity < 2; ++parity) {
        p.out = static_cast<char*>(out_full) + parity * pb;
        p.in = static_cast<const char*>(in_full) + (1 - parity) * pb;
        p.out_parity = parity;
        const int rc = launch_dslash(g, prec, recon, p, st);
        if (rc != TM_OK) return rc;
    }
    return TM_OK;
}

struct C44 {
    double re[4][4], im[4][4];
};
static C44 c44_mul(const C44& a, const C44& b)
{
    C44 c = {};
    for (int i = 0; i < 4; ++i)
        for (int j = 0; j < 4; ++j)
            for (int k = 0; k < 4; ++k) {
                c.re[i][j] += a.re[i][k] * b.re[k][j] - a.im[i][k] * b.im[k][j];
                c.im[i][j] += a.re[i][k] * b.im[k][j] + a.im[i][k] * b.re[k][j];
            }
    return c;
}

} // namespace tmk

using namespace tmk;

extern "C" int tm_covdev(const tm_lattice* L, const void* gauge, int prec, int recon, void* out_full, const void* in_full, int mu,
                         int nrhs, void* stream)
{
    if (!L || !gauge || !out_full || !in_full || !valid_prec(prec) || !valid_recon(recon)) return TM_ERR_ARG;
    if (out_full == in_full || mu < 0 || mu > 3 || nrhs < 1) return TM_ERR_ARG;
    if (!aligned256(gauge) || !aligned256(out_full) || !aligned256(in_full)) return TM_ERR_LAYOUT;
    cudaStream_t st = (cudaStream_t)stream;
    const Geo& g = L->g;
    recon = stored_recon(prec, recon);
    if (recon >= 100) return recon == 118 ? covdev_launch<2, 118>(g, gauge, out_full, in_full, mu, nrhs, st) : covdev_launch<2, 112>(g, gauge, out_full, in_full, mu, nrhs, st);
#define TM_COVDEV(P) (recon == 18 ? covdev_launch<P, 18>(g, gauge, out_full, in_full, mu, nrhs, st) : recon == 12 ? covdev_launch<P, 12>(g, gauge, out_full, in_full, mu, nrhs, st) : covdev_launch<P, 8>(g, gauge, out_full, in_full, mu, nrhs, st))
    if (prec == 8) return TM_COVDEV(8);
    if (prec == 4) return TM_COVDEV(4);
    return TM_COVDEV(2);
}

extern "C" int tm_contract_field(const tm_lattice* L, const void* a_full, const void* b_full, int prec, int nrhs, double* out,
                                 void* stream)
{
    if (!L || !a_full || !b_full || !out || !valid_prec(prec) || nrhs < 1) return TM_ERR_ARG;
    if (!aligned256(a_full) || !aligned256(b_full) || !aligned256(out)) return TM_ERR_LAYOUT;
    cudaStream_t st = (cudaStream_t)stream;
    const Geo& g = L->g;
    const size_t pb = spinor_parity_bytes(g, prec);
    dim3 grid((g.Vh + 127) / 128, 2, nrhs);
    if (prec == 8) contract_field_kernel<8><<<grid, 128, 0, st>>>(g, (const char*)a_full, (const char*)b_full, pb, out, L->V);
    else if (prec == 4) contract_field_kernel<4><<<grid, 128, 0, st>>>(g, (const char*)a_full, (const char*)b_full, pb, out, L->V);
    else contract_field_kernel<2><<<grid, 128, 0, st>>>(g, (const char*)a_full, (const char*)b_full, pb, out, L->V);
    TM_LAUNCH_CHECK("contract_field_kernel");
    return TM_OK;
}

extern "C" size_t tm_loop_momentum_workspace_bytes(const tm_lattice* L, int nrhs, int n_momenta, int pmax)
{
    if (!L || nrhs < 1 || n_momenta < 1 || pmax < 0 || pmax > MOM_MAXP) return 0;
    return round256((size_t)n_momenta * 3 * sizeof(int)) + mom_w2_bytes(L->g, pmax, nrhs);
}

extern "C" int tm_loop_momentum(const tm_lattice* L, const void* a_full, const void* b_full, int prec, int nrhs, const int* momenta,
                                int n_momenta, double* out, void* workspace, size_t workspace_bytes, void* stream)
{
    if (!L || !a_full || !b_full || !out || !workspace || !momenta || !valid_prec(prec) || nrhs < 1 || n_momenta < 1) return TM_ERR_ARG;
    if (!aligned256(a_full) || !aligned256(b_full) || !aligned256(out) || !aligned256(workspace)) return TM_ERR_LAYOUT;
    int P = 0;
    for (int i = 0; i < 3 * n_momenta; ++i) P = momenta[i] > P ? momenta[i] : (-momenta[i] > P ? -momenta[i] : P);
    if (P > MOM_MAXP) return TM_ERR_ARG;
    if (workspace_bytes < tm_loop_momentum_workspace_bytes(L, nrhs, n_momenta, P)) return TM_ERR_LAYOUT;
    const Geo& g = L->g;
    const size_t smem = mom_smem_bytes(g, P, prec);
    const int R = mom_rows(g);
    if (smem > 200 * 1024) return TM_ERR_LAYOUT;
    cudaStream_t st = (cudaStream_t)stream;
    int* mom_dev = static_cast<int*>(workspace);
    double2* W2 = reinterpret_cast<double2*>(static_cast<char*>(workspace) + round256((size_t)n_momenta * 3 * sizeof(int)));
    TM_CUDA_CHECK(cudaMemcpyAsync(mom_dev, momenta, (size_t)n_momenta * 3 * sizeof(int), cudaMemcpyHostToDevice, st));
    const size_t pb = spinor_parity_bytes(g, prec);
    dim3 grid(g.Z, g.T, nrhs);
    if (prec != 8 && g.X <= 64 && g.Y <= 128) {
        // fp32 / fp16 fields: warp-per-row kernel (no CTA barrier inside a plane, weights in the constant bank)
        MomWeights w;
        memset(&w, 0, sizeof(w));
        const double pi2 = 6.283185307179586476925286766559;
        for (int n = 0; n <= P; ++n)
            for (int j = 0; j < g.X / 2; ++j) {
                w.xc[n][j] = (float)cos(pi2 * ((n * j) % g.X) / g.X);
                w.xs[n][j] = (float)sin(pi2 * ((n * j) % g.X) / g.X);
            }
        for (int y = 0; y < g.Y; ++y)
            for (int m = 0; m <= P; ++m) {
                w.yw[y][m] = (float)cos(pi2 * ((m * y) % g.Y) / g.Y);
                if (m > 0) w.yw[y][P + m] = (float)sin(pi2 * ((m * y) % g.Y) / g.Y);
            }
        const int nwarp = (g.Y + MOMR_ROWS - 1) / MOMR_ROWS;
        const size_t NX = 2 * P + 1;
        const size_t tile_words = (size_t)(g.X > 32 ? 64 : 32) * 33, part_words = NX * NX * 32;
        const size_t rsmem = (size_t)nwarp * (tile_words > part_words ? tile_words : part_words) * sizeof(float);
#define TM_MOMR_GO(PR, PP, XH_, MAXT_, MINB_)                                                                                   \
    do {                                                                                                                        \
        TM_CUDA_CHECK(cudaFuncSetAttribute(loop_mom_row_kernel<PR, PP, XH_, MAXT_, MINB_>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rsmem)); \
        loop_mom_row_kernel<PR, PP, XH_, MAXT_, MINB_><<<grid, 32 * nwarp, rsmem, st>>>(g, (const char*)a_full, (const char*)b_full, pb, w, W2); \
    } while (0)
        // the 32^3 x 64 ensemble shape gets the unrolled x loop and CTAs of four warps; everything else the general form
#define TM_MOMR_LAUNCH(PR, PP)                                                                                                  \
    do {                                                                                                                        \
        if (g.X == 32 && nwarp <= 4) TM_MOMR_GO(PR, PP, 16, 128, MomrMinb<PR>::value);                                                  \
        else TM_MOMR_GO(PR, PP, 0, 512, 1);                                                                                     \
    } while (0)
#define TM_MOMR_SWITCH(PR)                                                                                                      \
    switch (P) {                                                                                                                \
    case 0: TM_MOMR_LAUNCH(PR, 0); break;                                                                                       \
    case 1: TM_MOMR_LAUNCH(PR, 1); break;                                                                                       \
    case 2: TM_MOMR_LAUNCH(PR, 2); break;                                                                                       \
    case 3: TM_MOMR_LAUNCH(PR, 3); break;                                                                                       \
    default: TM_MOMR_LAUNCH(PR, 4); break;                                                                                      \
    }
        if (prec == 4) {
            TM_MOMR_SWITCH(4)
        } else {
            TM_MOMR_SWITCH(2)
        }
        TM_LAUNCH_CHECK("loop_mom_row_kernel");
        static const GammaTable tbr = make_gamma_table();
        loop_mom_final_kernel<<<dim3(g.T, nrhs, (n_momenta + 7) / 8), 128, 0, st>>>(g, P, W2, mom_dev, n_momenta, tbr, out);
        TM_LAUNCH_CHECK("loop_mom_final_kernel");
        return TM_OK;
    }
#define TM_MOM_LAUNCH(PR, PP)                                                                                                   \
    do {                                                                                                                        \
        TM_CUDA_CHECK(cudaFuncSetAttribute(loop_mom_plane_kernel<PR, PP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
        loop_mom_plane_kernel<PR, PP><<<grid, MOM_THREADS, smem, st>>>(g, (const char*)a_full, (const char*)b_full, pb, R, W2);   \
    } while (0)
#define TM_MOM_SWITCH(PR)                                                                                                       \
    switch (P) {                                                                                                                \
    case 0: TM_MOM_LAUNCH(PR, 0); break;                                                                                        \
    case 1: TM_MOM_LAUNCH(PR, 1); break;                                                                                        \
    case 2: TM_MOM_LAUNCH(PR, 2); break;                                                                                        \
    case 3: TM_MOM_LAUNCH(PR, 3); break;                                                                                        \
    default: TM_MOM_LAUNCH(PR, 4); break;                                                                                       \
    }
    if (prec == 8) {
        TM_MOM_SWITCH(8)
    } else if (prec == 4) {
        TM_MOM_SWITCH(4)
    } else {
        TM_MOM_SWITCH(2)
    }
    TM_LAUNCH_CHECK("loop_mom_plane_kernel");
    static const GammaTable tb = make_gamma_table();
    loop_mom_final_kernel<<<dim3(g.T, nrhs, (n_momenta + 7) / 8), 128, 0, st>>>(g, P, W2, mom_dev, n_momenta, tb, out);
    TM_LAUNCH_CHECK("loop_mom_final_kernel");
    return TM_OK;
}

extern "C" int tm_time_dilute(const tm_lattice* L, const void* in_full, int prec, int nrhs, const unsigned char* keep_slice,
                              void* out_full, void* stream)
{
    if (!L || !in_full || !out_full || !keep_slice || !valid_prec(prec) || nrhs < 1) return TM_ERR_ARG;
    if (L->g.T > 512) return TM_ERR_LAYOUT;
    if (!aligned256(in_full) || !aligned256(out_full)) return TM_ERR_LAYOUT;
    TimeMask m = {};
    for (int t = 0; t < L->g.T; ++t)
        if (keep_slice[t]) m.bits[t >> 5] |= 1u << (t & 31);
    const Geo& g = L->g;
    const int nchunk = 24 * prec / 16;
    dim3 grid((g.Vh + 255) / 256, 2 * nrhs);
    time_dilute_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(g, (const char*)in_full, (char*)out_full, spinor_parity_bytes(g, prec),
                                                               nchunk, prec == 2, m);
    TM_LAUNCH_CHECK("time_dilute_kernel");
    return TM_OK;
}

extern "C" int tm_hpe_remainder(const tm_lattice* L, const void* gauge, int prec, int recon, void* out_full, const void* s_full,
                                void* tmp_full, double kappa, double mu, int nrhs, void* stream)
{
    if (!L || !gauge || !out_full || !s_full || !tmp_full || !valid_prec(prec) || !valid_recon(recon)) return TM_ERR_ARG;
    if (out_full == s_full || tmp_full == s_full || tmp_full == out_full || nrhs < 1 || nrhs > TM_MAX_NRHS) return TM_ERR_ARG;
    if (!aligned256(gauge) || !aligned256(out_full) || !aligned256(s_full) || !aligned256(tmp_full)) return TM_ERR_LAYOUT;
    cudaStream_t st = (cudaStream_t)stream;
    const Geo& g = L->g;
    int rc = hpe_BH(g, gauge, prec, recon, tmp_full, s_full, kappa, mu, nrhs, st);
    if (rc == TM_OK) rc = hpe_BH(g, gauge, prec, recon, out_full, tmp_full, kappa, mu, nrhs, st);
    if (rc == TM_OK) rc = hpe_BH(g, gauge, prec, recon, tmp_full, out_full, kappa, mu, nrhs, st);
    if (rc == TM_OK) rc = hpe_BH(g, gauge, prec, recon, out_full, tmp_full, kappa, mu, nrhs, st);
    return rc;
}

extern "C" int tm_hpe_local_traces(double kappa, double mu, double* out16)
{
    if (!out16) return TM_ERR_ARG;
    // host arithmetic on 4x4 complex matrices: S = B + kappa^2 sum_mu [B (1-g) B (1+g) B + B (1+g) B (1-g) B], B = R^-1
    const double a = 2.0 * kappa * mu, d = 1.0 / (1.0 + a * a);
    GammaZ gm[4][4][4];
    gamma_mu_table(gm);
    C44 B = {};
    for (int i = 0; i < 4; ++i) {
        B.re[i][i] = d;
        B.im[i][i] = (i < 2 ? -a : a) * d; // (1 - i a g5)/(1 + a^2), g5 = diag(1,1,-1,-1)
    }
    C44 S = B;
    for (int m = 0; m < 4; ++m)
        for (int sg = -1; sg <= 1; sg += 2) {
            C44 Pm = {}, Pp = {};
            for (int i = 0; i < 4; ++i)
                for (int j = 0; j < 4; ++j) {
                    Pm.re[i][j] = (i == j) - sg * gm[m][i][j].re;
                    Pm.im[i][j] = -sg * gm[m][i][j].im;
                    Pp.re[i][j] = (i == j) + sg * gm[m][i][j].re;
                    Pp.im[i][j] = sg * gm[m][i][j].im;
                }
            const C44 t = c44_mul(c44_mul(c44_mul(c44_mul(B, Pm), B), Pp), B);
            for (int i = 0; i < 4; ++i)
                for (int j = 0; j < 4; ++j) {
                    S.re[i][j] += kappa * kappa * t.re[i][j];
                    S.im[i][j] += kappa * kappa * t.im[i][j];
                }
        }
    const GammaTable tb = make_gamma_table();
    for (int n = 0; n < 16; ++n) {
        double re = 0.0, im = 0.0; // 3 tr[Gamma_n S] = 3 sum_al Gamma_n[al][col] S[col][al]
        for (int al = 0; al < 4; ++al) {
            const int be = tb.col[n][al];
            re += tb.re[n][al] * S.re[be][al] - tb.im[n][al] * S.im[be][al];
            im += tb.re[n][al] * S.im[be][al] + tb.im[n][al] * S.re[be][al];
        }
        out16[2 * n] = 3.0 * re;
        out16[2 * n + 1] = 3.0 * im;
    }
    return TM_OK;
}
