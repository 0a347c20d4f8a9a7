// tm_dslash_tile.cuh -- fp32 / fp16-storage hopping term, one thread per (site, right-hand side)
// (SURVEY.md 8(a) rows a2, a3, a7; PAPER.md:384 fused kernels, :403 link reconstruction).
//
//   out = (p0 + i p1 g5) x + (q0 + i q1 g5) sum_mu [(1-g_mu) s U_mu(x) in(x+mu) + (1+g_mu) s U_mu(x-mu)^dag in(x-mu)]
//
// CTA = S consecutive checkerboard sites (threadIdx.x) x RB right-hand sides (threadIdx.y); a warp is 32 sites
// of ONE right-hand side, so every spinor access is a fully coalesced 128-bit load.
//   phase A (SL = links through shared memory, used when nrhs > 1): the CTA's 8*S links are loaded once,
//     converted to fp32, rebuilt from 12 reals, daggered for the backward hops, multiplied by the antiperiodic
//     sign and parked in shared memory; the 8 neighbour indices of every site go there too.  All RB right-hand
//     sides of the tile reuse them ("reuses each gauge link load", BASELINE.json north_star).
//   phase B: per direction: raw 16-byte chunks of the neighbour -> spin
//     projection to a half spinor (12 reals) -> SU(3) multiply -> reconstruction into the accumulator.
// fp16 storage: the projection adds the binary16 words directly in fp32 (FHADD: f32 = f16 + f32, exact
// inputs), and the per-site norm multiplies the 12 projected-and-rotated reals inside the reconstruction FMAs
// instead of the 24 loaded ones.  The dagger is a template parameter: all signs are instruction modifiers.
#pragma once
#include "tm_dslash.cuh"

namespace tmk {

// ---- raw (unconverted) site data --------------------------------------------------------------------
template <int PREC> struct Raw;
template <> struct Raw<4> {
    float4 q[6];
};
template <> struct Raw<2> {
    uint4 q[3];
    float nrm;
};

template <int PREC>
__device__ __forceinline__ void load_raw(const void* base, int Vh, int cb, Raw<PREC>& r)
{
    if constexpr (PREC == 4) {
        const float4* p = reinterpret_cast<const float4*>(base) + cb;
#pragma unroll
        for (int k = 0; k < 6; ++k) r.q[k] = __ldg(p + (size_t)k * Vh);
    } else {
        const uint4* p = reinterpret_cast<const uint4*>(base) + cb;
#pragma unroll
        for (int k = 0; k < 3; ++k) r.q[k] = __ldg(p + (size_t)k * Vh);
        r.nrm = __ldg(reinterpret_cast<const float*>(reinterpret_cast<const uint4*>(base) + (size_t)3 * Vh) + cb);
    }
}

// binary16 word (re = low half, im = high half) helpers; FHADD takes the half select and the sign as modifiers
__device__ __forceinline__ float h_lo(uint32_t w)
{
    float r;
    asm("{.reg .b16 l,h; mov.b32 {l,h}, %1; cvt.f32.f16 %0, l;}" : "=f"(r) : "r"(w));
    return r;
}
__device__ __forceinline__ float h_hi(uint32_t w)
{
    float r;
    asm("{.reg .b16 l,h; mov.b32 {l,h}, %1; cvt.f32.f16 %0, h;}" : "=f"(r) : "r"(w));
    return r;
}
// c + sign * (half HI ? high : low of w), sign = NEG ? -1 : +1
template <int HI, int NEG>
__device__ __forceinline__ float h_add(uint32_t w, float c)
{
    float r;
    if (HI && NEG) asm("{.reg .b16 l,h; mov.b32 {l,h}, %1; neg.f16 h, h; add.rn.f32.f16 %0, h, %2;}" : "=f"(r) : "r"(w), "f"(c));
    if (HI && !NEG) asm("{.reg .b16 l,h; mov.b32 {l,h}, %1; add.rn.f32.f16 %0, h, %2;}" : "=f"(r) : "r"(w), "f"(c));
    if (!HI && NEG) asm("{.reg .b16 l,h; mov.b32 {l,h}, %1; neg.f16 l, l; add.rn.f32.f16 %0, l, %2;}" : "=f"(r) : "r"(w), "f"(c));
    if (!HI && !NEG) asm("{.reg .b16 l,h; mov.b32 {l,h}, %1; add.rn.f32.f16 %0, l, %2;}" : "=f"(r) : "r"(w), "f"(c));
    return r;
}

// complex number (spin s, colour c) of a raw site: accessors for both storage types
template <int PREC>
struct Cx {
    // fp32: value pair; fp16: the packed word
    float re, im;
    uint32_t w;
};
template <int PREC>
__device__ __forceinline__ Cx<PREC> raw_cx(const Raw<PREC>& r, int j) // j = s*3 + c, compile-time after unrolling
{
    Cx<PREC> z;
    if constexpr (PREC == 4) {
        const float4 q = r.q[j >> 1];
        z.re = (j & 1) ? q.z : q.x;
        z.im = (j & 1) ? q.w : q.y;
        z.w = 0;
    } else {
        const uint4 q = r.q[j >> 2];
        z.w = (j & 3) == 0 ? q.x : (j & 3) == 1 ? q.y : (j & 3) == 2 ? q.z : q.w;
        z.re = z.im = 0;
    }
    return z;
}
// h = a + SG * b
template <int PREC, int SG>
__device__ __forceinline__ void cx_add(const Cx<PREC>& a, const Cx<PREC>& b, float& hr, float& hi)
{
    if constexpr (PREC == 4) {
        hr = SG > 0 ? a.re + b.re : a.re - b.re;
        hi = SG > 0 ? a.im + b.im : a.im - b.im;
    } else {
        hr = h_add<0, (SG < 0)>(b.w, h_lo(a.w));
        hi = h_add<1, (SG < 0)>(b.w, h_hi(a.w));
    }
}
// h = a + SG * i * b  : hr = ar - SG bi ; hi = ai + SG br
template <int PREC, int SG>
__device__ __forceinline__ void cx_addi(const Cx<PREC>& a, const Cx<PREC>& b, float& hr, float& hi)
{
    if constexpr (PREC == 4) {
        hr = SG > 0 ? a.re - b.im : a.re + b.im;
        hi = SG > 0 ? a.im + b.re : a.im - b.re;
    } else {
        hr = h_add<1, (SG > 0)>(b.w, h_lo(a.w));
        hi = h_add<0, (SG < 0)>(b.w, h_hi(a.w));
    }
}

// h[12] = upper half of (1 - E g_mu) psi (un-normalised for fp16: the site norm is applied in tile_reconstruct)
template <int PREC, int MU, int E>
__device__ __forceinline__ void tile_project(const Raw<PREC>& r, float* h)
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const Cx<PREC> p0 = raw_cx<PREC>(r, c), p1 = raw_cx<PREC>(r, 3 + c), p2 = raw_cx<PREC>(r, 6 + c), p3 = raw_cx<PREC>(r, 9 + c);
        if (MU == 0) { // h0 = p0 + E i p3 ; h1 = p1 + E i p2
            cx_addi<PREC, E>(p0, p3, h[2 * c], h[2 * c + 1]);
            cx_addi<PREC, E>(p1, p2, h[6 + 2 * c], h[6 + 2 * c + 1]);
        } else if (MU == 1) { // h0 = p0 + E p3 ; h1 = p1 - E p2
            cx_add<PREC, E>(p0, p3, h[2 * c], h[2 * c + 1]);
            cx_add<PREC, -E>(p1, p2, h[6 + 2 * c], h[6 + 2 * c + 1]);
        } else if (MU == 2) { // h0 = p0 + E i p2 ; h1 = p1 - E i p3
            cx_addi<PREC, E>(p0, p2, h[2 * c], h[2 * c + 1]);
            cx_addi<PREC, -E>(p1, p3, h[6 + 2 * c], h[6 + 2 * c + 1]);
        } else { // h0 = p0 - E p2 ; h1 = p1 - E p3
            cx_add<PREC, -E>(p0, p2, h[2 * c], h[2 * c + 1]);
            cx_add<PREC, -E>(p1, p3, h[6 + 2 * c], h[6 + 2 * c + 1]);
        }
    }
}

// acc += w * (g, lower(g)), lower rebuilt from the upper half; w = site norm (fp16) or absent (fp32)
template <int MU, int E, bool SCALED>
__device__ __forceinline__ void tile_reconstruct(float* acc, const float* g, float w)
{
    const float wp = SCALED ? w : 1.f;
    const float we = (E > 0) ? wp : -wp; // E * w
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float g0r = g[2 * c], g0i = g[2 * c + 1], g1r = g[6 + 2 * c], g1i = g[6 + 2 * c + 1];
        acc[2 * c] = fmaf(wp, g0r, acc[2 * c]);
        acc[2 * c + 1] = fmaf(wp, g0i, acc[2 * c + 1]);
        acc[6 + 2 * c] = fmaf(wp, g1r, acc[6 + 2 * c]);
        acc[6 + 2 * c + 1] = fmaf(wp, g1i, acc[6 + 2 * c + 1]);
        if (MU == 0) { // lower = (-E i g1, -E i g0)
            acc[12 + 2 * c] = fmaf(we, g1i, acc[12 + 2 * c]);
            acc[12 + 2 * c + 1] = fmaf(-we, g1r, acc[12 + 2 * c + 1]);
            acc[18 + 2 * c] = fmaf(we, g0i, acc[18 + 2 * c]);
            acc[18 + 2 * c + 1] = fmaf(-we, g0r, acc[18 + 2 * c + 1]);
        } else if (MU == 1) { // lower = (-E g1, E g0)
            acc[12 + 2 * c] = fmaf(-we, g1r, acc[12 + 2 * c]);
            acc[12 + 2 * c + 1] = fmaf(-we, g1i, acc[12 + 2 * c + 1]);
            acc[18 + 2 * c] = fmaf(we, g0r, acc[18 + 2 * c]);
            acc[18 + 2 * c + 1] = fmaf(we, g0i, acc[18 + 2 * c + 1]);
        } else if (MU == 2) { // lower = (-E i g0, E i g1)
            acc[12 + 2 * c] = fmaf(we, g0i, acc[12 + 2 * c]);
            acc[12 + 2 * c + 1] = fmaf(-we, g0r, acc[12 + 2 * c + 1]);
            acc[18 + 2 * c] = fmaf(-we, g1i, acc[18 + 2 * c]);
            acc[18 + 2 * c + 1] = fmaf(we, g1r, acc[18 + 2 * c + 1]);
        } else { // lower = (-E g0, -E g1)
            acc[12 + 2 * c] = fmaf(-we, g0r, acc[12 + 2 * c]);
            acc[12 + 2 * c + 1] = fmaf(-we, g0i, acc[12 + 2 * c + 1]);
            acc[18 + 2 * c] = fmaf(-we, g1r, acc[18 + 2 * c]);
            acc[18 + 2 * c + 1] = fmaf(-we, g1i, acc[18 + 2 * c + 1]);
        }
    }
}

// neighbour indices of checkerboard site cb (order: +x -x +y -y +z -z +t -t) and the two temporal hop signs
__device__ __forceinline__ void tile_neighbours(const Geo& g, int parity, int cb, int* nb, float& sgp, float& sgm)
{
    uint32_t t, rem, z, rem2, y, xh;
    g.dXh.divmod((uint32_t)cb, rem, xh);
    g.dY.divmod(rem, rem2, y);
    g.dZ.divmod(rem2, t, z);
    const int xodd = (parity + y + z + t) & 1;
    const int Xh = g.Xh, XhY = g.XhY, V3h = g.V3h, Vh = g.Vh;
    nb[0] = cb + (xodd ? ((int)xh == Xh - 1 ? 1 - Xh : 1) : 0);
    nb[1] = cb - (xodd ? 0 : ((int)xh == 0 ? 1 - Xh : 1));
    nb[2] = cb + ((int)y == g.Y - 1 ? Xh - XhY : Xh);
    nb[3] = cb - ((int)y == 0 ? Xh - XhY : Xh);
    nb[4] = cb + ((int)z == g.Z - 1 ? XhY - V3h : XhY);
    nb[5] = cb - ((int)z == 0 ? XhY - V3h : XhY);
    nb[6] = cb + ((int)t == g.T - 1 ? V3h - Vh : V3h);
    nb[7] = cb - ((int)t == 0 ? V3h - Vh : V3h);
    sgp = (g.ap && (int)t == g.T - 1) ? -1.f : 1.f;
    sgm = (g.ap && (int)t == 0) ? -1.f : 1.f;
}

template <int S>
struct TileSmem {
    int nbr[8][S];
    float4 u4[8][4][S];
    float2 u2[8][S];
};

// fused epilogue of one (site, rhs): out = (p0 + i p1 g5) x + (q0 + i q1 g5) acc ; g5 = diag(1,1,-1,-1); optional residual
// update, store, optional reduction partial
template <int PREC>
__device__ __forceinline__ void tile_epilogue(const DslashKArgs& a, int cb, int rhs, const float* acc)
{
    const int Vh = a.g.Vh;
    const float p0 = (float)a.pq[0], p1 = (float)a.pq[1], q0 = (float)a.pq[2], q1 = (float)a.pq[3];
    float o[24];
#pragma unroll
    for (int k = 0; k < 12; ++k) {
        const float s5 = (k < 6) ? 1.f : -1.f;
        const float dr = acc[2 * k], di = acc[2 * k + 1];
        // explicit operation order: the packed variant (tile_site2) rounds identically, so a right-hand side gives the same
        // bits whether it runs alone or in a batch
        o[2 * k] = fmaf(-s5 * q1, di, q0 * dr);
        o[2 * k + 1] = fmaf(s5 * q1, dr, q0 * di);
    }
    if (a.x != nullptr) {
        float xv[24];
        load_spinor<PREC, 1>(a.x + (size_t)rhs * a.stride_x, Vh, cb, xv);
#pragma unroll
        for (int k = 0; k < 12; ++k) {
            const float s5 = (k < 6) ? 1.f : -1.f;
            o[2 * k] = fmaf(-s5 * p1, xv[2 * k + 1], fmaf(p0, xv[2 * k], o[2 * k]));
            o[2 * k + 1] = fmaf(s5 * p1, xv[2 * k], fmaf(p0, xv[2 * k + 1], o[2 * k + 1]));
        }
    }
    if (a.axpy_y != nullptr) fused_axpy<PREC>(a, rhs, cb, o);
    store_spinor<PREC>(a.out + (size_t)rhs * a.stride_out, Vh, cb, o);
    if (a.dot_partial != nullptr) warp_dot_store<PREC>(a, rhs, cb, o);
}


// phase B + epilogue for one (site cb, right-hand side rhs): 8 hops from the neighbours nb[8], fused epilogue, store.
// SL != 0: links come from the tile image `sm` (lane tx), already daggered and signed; SL == 0: loaded per thread.
template <int PREC, int RECON, int DAG, int SL, typename SM>
__device__ __forceinline__ void tile_site(const DslashKArgs& a, const SM& sm, int cb, int tx, int rhs, const int* nb, float sgp,
                                          float sgm)
{
    constexpr int E = DAG ? -1 : 1;
    constexpr bool SC = (PREC == 2);
    const int Vh = a.g.Vh;
    const char* in = a.in + (size_t)rhs * a.stride_in;
    float acc[24];
#pragma unroll
    for (int k = 0; k < 24; ++k) acc[k] = 0.f;

    Raw<PREC> cur;
#pragma unroll
    for (int d = 0; d < 8; ++d) {
#ifdef TM_DEBUG_NOLDG // timing ablation (probe builds only, wrong results): no gather, the raw words come from registers
        {
            unsigned* w_ = reinterpret_cast<unsigned*>(&cur);
#pragma unroll
            for (int k = 0; k < (int)(sizeof(cur) / 4); ++k) w_[k] = 0x3c003800u + (unsigned)((nb[d] + k) & 0x3ff);
            if constexpr (PREC == 2) cur.nrm = __int_as_float(0x3f800000 + (nb[d] & 0xffff));
        }
#else
        load_raw<PREC>(in, Vh, nb[d], cur); // (a register prefetch of direction d + 1 was measured: no gain at 80 / 128 registers)
#endif
        float u[18];
#ifdef TM_DEBUG_NOLDS // timing ablation (probe builds only, wrong results): no shared-memory link read
        if constexpr (SL) {
#pragma unroll
            for (int k = 0; k < 18; ++k) u[k] = __int_as_float(0x3f000000 + nb[d] * 32 + k);
        } else
#endif
        if constexpr (SL) {
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const float4 q = sm.u4[d][k][tx];
                u[4 * k] = q.x;
                u[4 * k + 1] = q.y;
                u[4 * k + 2] = q.z;
                u[4 * k + 3] = q.w;
            }
            const float2 q2 = sm.u2[d][tx];
            u[16] = q2.x;
            u[17] = q2.y;
        } else {
            const bool fwd = !(d & 1);
            const char* blk = a.gauge + (size_t)((fwd ? a.parity : 1 - a.parity) * 4 + (d >> 1)) * a.link_block;
            load_link<PREC, RECON>(blk, Vh, fwd ? cb : nb[d], u);
        }
        float h[12], g[12];
        float w = 1.f;
        if constexpr (SC) w = cur.nrm;
        // direction d = 2*mu + (backward): projector sign E for forward, -E for backward
        if (d == 0) tile_project<PREC, 0, E>(cur, h);
        if (d == 1) tile_project<PREC, 0, -E>(cur, h);
        if (d == 2) tile_project<PREC, 1, E>(cur, h);
        if (d == 3) tile_project<PREC, 1, -E>(cur, h);
        if (d == 4) tile_project<PREC, 2, E>(cur, h);
        if (d == 5) tile_project<PREC, 2, -E>(cur, h);
        if (d == 6) tile_project<PREC, 3, E>(cur, h);
        if (d == 7) tile_project<PREC, 3, -E>(cur, h);
        if constexpr (SL) {
            su3_mul<0>(u, h, g);
        } else {
            if (d & 1) su3_mul<1>(u, h, g);
            else su3_mul<0>(u, h, g);
            if (d == 6) w *= sgp;
            if (d == 7) w *= sgm;
        }
        if (d == 0) tile_reconstruct<0, E, true>(acc, g, w);
        if (d == 1) tile_reconstruct<0, -E, true>(acc, g, w);
        if (d == 2) tile_reconstruct<1, E, true>(acc, g, w);
        if (d == 3) tile_reconstruct<1, -E, true>(acc, g, w);
        if (d == 4) tile_reconstruct<2, E, true>(acc, g, w);
        if (d == 5) tile_reconstruct<2, -E, true>(acc, g, w);
        if (d == 6) tile_reconstruct<3, E, true>(acc, g, w);
        if (d == 7) tile_reconstruct<3, -E, true>(acc, g, w);
    }

    tile_epilogue<PREC>(a, cb, rhs, acc);
}

// ---- packed fp32x2 variant of phase B ----------------------------------------------------------------
// sm_100a issues `fma.rn.f32x2` (SASS FFMA2: two fp32 FMAs on a 64-bit register pair, one issue slot, scalar operands
// broadcast and negated as modifiers).  The two spin components of a projected half spinor are multiplied by the SAME
// link, so they form the pair: H[k] = (h_spin0[k], h_spin1[k]), k = 2*colour + reim.  The SU(3) product is then 36 FFMA2
// instead of 72 FFMA per direction, the reconstruction 12 instead of 24, with the same rounding per real as the scalar
// code (each lane is an IEEE fp32 FMA).  Accumulators: AU[k] = (acc[k], acc[6+k]) (spins 0,1); the lower spins are kept
// as (spin3, spin2) while mu = x,y are processed (their reconstruction crosses the spins) and as (spin2, spin3)
// afterwards; the swap is folded into the scalar FMAs of the first z hop.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float lo, float hi)
{
    f32x2 r;
    asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void upk2(f32x2 p, float& lo, float& hi) { asm("mov.b64 {%0,%1}, %2;" : "=f"(lo), "=f"(hi) : "l"(p)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 bc2(float s) { return pk2(s, s); } // ptxas folds this into a scalar-broadcast operand

// G = U H for both spins at once; u row-major complex 3x3 (DAG: the adjoint is applied)
template <int DAG>
__device__ __forceinline__ void su3_mul2(const float* u, const f32x2* H, f32x2* G)
{
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        f32x2 re, im;
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const float ur = DAG ? u[2 * (b * 3 + a)] : u[2 * (a * 3 + b)];
            const float ui = DAG ? -u[2 * (b * 3 + a) + 1] : u[2 * (a * 3 + b) + 1];
            if (b == 0) {
                re = mul2(bc2(ur), H[0]);
                im = mul2(bc2(ur), H[1]);
            } else {
                re = fma2(bc2(ur), H[2 * b], re);
                im = fma2(bc2(ur), H[2 * b + 1], im);
            }
            re = fma2(bc2(-ui), H[2 * b + 1], re);
            im = fma2(bc2(ui), H[2 * b], im);
        }
        G[2 * a] = re;
        G[2 * a + 1] = im;
    }
}

// AU += w G; lower spins from the upper ones.  MU 0,1 update AL in (spin3, spin2) order, MU 2,3 in (spin2, spin3) order;
// SWAPIN: AL arrives in (spin3, spin2) order and leaves in (spin2, spin3) order (first hop of mu = 2).
template <int MU, int E, bool FIRST, bool SWAPIN>
__device__ __forceinline__ void tile_reconstruct2(f32x2* AU, f32x2* AL, const f32x2* G, float w)
{
    const float we = (E > 0) ? w : -w;
#pragma unroll
    for (int k = 0; k < 6; ++k) AU[k] = FIRST ? mul2(bc2(w), G[k]) : fma2(bc2(w), G[k], AU[k]);
    if (MU == 0) { // lower = (-E i g1, -E i g0): (spin3, spin2) re += we (g0i, g1i), im += -we (g0r, g1r)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            AL[2 * c] = FIRST ? mul2(bc2(we), G[2 * c + 1]) : fma2(bc2(we), G[2 * c + 1], AL[2 * c]);
            AL[2 * c + 1] = FIRST ? mul2(bc2(-we), G[2 * c]) : fma2(bc2(-we), G[2 * c], AL[2 * c + 1]);
        }
    } else if (MU == 1) { // lower = (-E g1, E g0): (spin3, spin2) += (we g0, -we g1)
        const f32x2 pm = pk2(we, -we);
#pragma unroll
        for (int k = 0; k < 6; ++k) AL[k] = fma2(pm, G[k], AL[k]);
    } else if (MU == 2) { // lower = (-E i g0, E i g1): (spin2, spin3) re += (we g0i, -we g1i), im += (-we g0r, we g1r)
        if (SWAPIN) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                float s3, s2, gl, gh;
                upk2(AL[2 * c], s3, s2);
                upk2(G[2 * c + 1], gl, gh);
                AL[2 * c] = pk2(fmaf(we, gl, s2), fmaf(-we, gh, s3));
                upk2(AL[2 * c + 1], s3, s2);
                upk2(G[2 * c], gl, gh);
                AL[2 * c + 1] = pk2(fmaf(-we, gl, s2), fmaf(we, gh, s3));
            }
        } else {
            const f32x2 pm = pk2(we, -we), mp = pk2(-we, we);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                AL[2 * c] = fma2(pm, G[2 * c + 1], AL[2 * c]);
                AL[2 * c + 1] = fma2(mp, G[2 * c], AL[2 * c + 1]);
            }
        }
    } else { // lower = (-E g0, -E g1)
#pragma unroll
        for (int k = 0; k < 6; ++k) AL[k] = fma2(bc2(-we), G[k], AL[k]);
    }
}

template <int PREC, int RECON, int DAG, int SL, typename SM>
__device__ __forceinline__ void tile_site2(const DslashKArgs& a, const SM& sm, int cb, int tx, int rhs, const int* nb, float sgp,
                                           float sgm)
{
    constexpr int E = DAG ? -1 : 1;
    const int Vh = a.g.Vh;
    const char* in = a.in + (size_t)rhs * a.stride_in;
    f32x2 AU[6], AL[6];

    Raw<PREC> cur;
#pragma unroll
    for (int d = 0; d < 8; ++d) {
        load_raw<PREC>(in, Vh, nb[d], cur);
        float u[18];
        if constexpr (SL) {
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const float4 q = sm.u4[d][k][tx];
                u[4 * k] = q.x;
                u[4 * k + 1] = q.y;
                u[4 * k + 2] = q.z;
                u[4 * k + 3] = q.w;
            }
            const float2 q2 = sm.u2[d][tx];
            u[16] = q2.x;
            u[17] = q2.y;
        } else {
            const bool fwd = !(d & 1);
            const char* blk = a.gauge + (size_t)((fwd ? a.parity : 1 - a.parity) * 4 + (d >> 1)) * a.link_block;
            // temporal gauge declared (RECON = reals + 200): a temporal hop that does not wrap around crosses a unit link
            const bool unit_hop = RECON >= 200 && ((d == 6 && nb[6] > cb) || (d == 7 && nb[7] < cb));
#ifdef TM_DEBUG_LINKWIN // timing ablation (probe builds only, wrong results): every link load lands in a 1024-site window (L1 / L2 hits)
            if (!unit_hop) load_link<PREC, RECON>(blk, Vh, (fwd ? cb : nb[d]) & 1023, u);
#else
            if (!unit_hop) load_link<PREC, RECON>(blk, Vh, fwd ? cb : nb[d], u);
#endif
        }
        float h[12];
        float w = 1.f;
        if constexpr (PREC == 2) w = cur.nrm;
        if (d == 0) tile_project<PREC, 0, E>(cur, h);
        if (d == 1) tile_project<PREC, 0, -E>(cur, h);
        if (d == 2) tile_project<PREC, 1, E>(cur, h);
        if (d == 3) tile_project<PREC, 1, -E>(cur, h);
        if (d == 4) tile_project<PREC, 2, E>(cur, h);
        if (d == 5) tile_project<PREC, 2, -E>(cur, h);
        if (d == 6) tile_project<PREC, 3, E>(cur, h);
        if (d == 7) tile_project<PREC, 3, -E>(cur, h);
        f32x2 H[6], G[6];
#pragma unroll
        for (int k = 0; k < 6; ++k) H[k] = pk2(h[k], h[6 + k]);
        if constexpr (SL) {
            su3_mul2<0>(u, H, G);
        } else {
            if (RECON >= 200 && ((d == 6 && nb[6] > cb) || (d == 7 && nb[7] < cb))) {
#pragma unroll
                for (int k = 0; k < 6; ++k) G[k] = H[k];
            } else if (d & 1) {
                su3_mul2<1>(u, H, G);
            } else {
                su3_mul2<0>(u, H, G);
            }
            if (d == 6) w *= sgp;
            if (d == 7) w *= sgm;
        }
        if (d == 0) tile_reconstruct2<0, E, true, false>(AU, AL, G, w);
        if (d == 1) tile_reconstruct2<0, -E, false, false>(AU, AL, G, w);
        if (d == 2) tile_reconstruct2<1, E, false, false>(AU, AL, G, w);
        if (d == 3) tile_reconstruct2<1, -E, false, false>(AU, AL, G, w);
        if (d == 4) tile_reconstruct2<2, E, false, true>(AU, AL, G, w);
        if (d == 5) tile_reconstruct2<2, -E, false, false>(AU, AL, G, w);
        if (d == 6) tile_reconstruct2<3, E, false, false>(AU, AL, G, w);
        if (d == 7) tile_reconstruct2<3, -E, false, false>(AU, AL, G, w);
    }

    // epilogue: out = (p0 + i p1 g5) x + (q0 + i q1 g5) acc ; g5 = diag(1,1,-1,-1); pairs: AU = spins (0,1), AL = spins (2,3)
    const float p0 = (float)a.pq[0], p1 = (float)a.pq[1], q0 = (float)a.pq[2], q1 = (float)a.pq[3];
    f32x2 OU[6], OL[6];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        OU[2 * c] = fma2(bc2(-q1), AU[2 * c + 1], mul2(bc2(q0), AU[2 * c]));
        OU[2 * c + 1] = fma2(bc2(q1), AU[2 * c], mul2(bc2(q0), AU[2 * c + 1]));
        OL[2 * c] = fma2(bc2(q1), AL[2 * c + 1], mul2(bc2(q0), AL[2 * c]));
        OL[2 * c + 1] = fma2(bc2(-q1), AL[2 * c], mul2(bc2(q0), AL[2 * c + 1]));
    }
    if (a.x != nullptr) {
        float xv[24];
        load_spinor<PREC, 1>(a.x + (size_t)rhs * a.stride_x, Vh, cb, xv);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const f32x2 xur = pk2(xv[2 * c], xv[6 + 2 * c]), xui = pk2(xv[2 * c + 1], xv[6 + 2 * c + 1]);
            const f32x2 xlr = pk2(xv[12 + 2 * c], xv[18 + 2 * c]), xli = pk2(xv[12 + 2 * c + 1], xv[18 + 2 * c + 1]);
            OU[2 * c] = fma2(bc2(-p1), xui, fma2(bc2(p0), xur, OU[2 * c]));
            OU[2 * c + 1] = fma2(bc2(p1), xur, fma2(bc2(p0), xui, OU[2 * c + 1]));
            OL[2 * c] = fma2(bc2(p1), xli, fma2(bc2(p0), xlr, OL[2 * c]));
            OL[2 * c + 1] = fma2(bc2(-p1), xlr, fma2(bc2(p0), xli, OL[2 * c + 1]));
        }
    }
    float o[24];
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        upk2(OU[k], o[k], o[6 + k]);
        upk2(OL[k], o[12 + k], o[18 + k]);
    }
    if (a.axpy_y != nullptr) fused_axpy<PREC>(a, rhs, cb, o);
    store_spinor<PREC>(a.out + (size_t)rhs * a.stride_out, Vh, cb, o);
    if (a.dot_partial != nullptr) warp_dot_store<PREC>(a, rhs, cb, o);
}

#ifndef TM_F2
#define TM_F2 1
#endif
template <int PREC, int RECON, int DAG, int SL, typename SM>
__device__ __forceinline__ void tile_site_any(const DslashKArgs& a, const SM& sm, int cb, int tx, int rhs, const int* nb, float sgp,
                                              float sgm)
{
    // measured on B200: the packed form is 8-10 % faster where every thread also loads, converts and
    // rebuilds its own links (nrhs = 1) and 5 % slower in the multi-rhs kernels, whose FMA and LSU pipes are already balanced
    static_assert(RECON < 200 || (TM_F2 == 1 && SL == 0), "the temporal-gauge codes exist for the packed single-rhs form");
    if constexpr (TM_F2 == 1 ? SL == 0 : TM_F2 == 2) tile_site2<PREC, RECON, DAG, SL>(a, sm, cb, tx, rhs, nb, sgp, sgm);
    else tile_site<PREC, RECON, DAG, SL>(a, sm, cb, tx, rhs, nb, sgp, sgm);
}

// phase A for one tile: neighbour indices (the antiperiodic sign of a temporal hop rides on the index as ~index) and the
// 8*S links as fp32, rebuilt, daggered for backward hops, signed.  All `nthreads` threads of the CTA call it.
template <int PREC, int RECON, int S>
__device__ __forceinline__ void tile_build(const DslashKArgs& a, int cb0, int tid, int nthreads, TileSmem<S>& sm)
{
    const int Vh = a.g.Vh;
    if (tid < S && cb0 + tid < Vh) {
        int nb[8];
        float sgp, sgm;
        tile_neighbours(a.g, a.parity, cb0 + tid, nb, sgp, sgm);
#pragma unroll
        for (int d = 0; d < 8; ++d) sm.nbr[d][tid] = (d == 6 && sgp < 0.f) || (d == 7 && sgm < 0.f) ? ~nb[d] : nb[d];
    }
    __syncthreads();
    for (int l = tid; l < 8 * S; l += nthreads) {
        const int d = l / S, s = l - d * S;
        if (cb0 + s >= Vh) continue;
        const bool fwd = !(d & 1);
        int nbi = sm.nbr[d][s];
        const float sg = nbi < 0 ? -1.f : 1.f;
        nbi = nbi < 0 ? ~nbi : nbi;
        const char* blk = a.gauge + (size_t)((fwd ? a.parity : 1 - a.parity) * 4 + (d >> 1)) * a.link_block;
        float u[18];
        load_link<PREC, RECON>(blk, Vh, fwd ? cb0 + s : nbi, u);
        float w[18];
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                w[2 * (i * 3 + j)] = sg * (fwd ? u[2 * (i * 3 + j)] : u[2 * (j * 3 + i)]);
                w[2 * (i * 3 + j) + 1] = sg * (fwd ? u[2 * (i * 3 + j) + 1] : -u[2 * (j * 3 + i) + 1]);
            }
#pragma unroll
        for (int k = 0; k < 4; ++k) sm.u4[d][k][s] = make_float4(w[4 * k], w[4 * k + 1], w[4 * k + 2], w[4 * k + 3]);
        sm.u2[d][s] = make_float2(w[16], w[17]);
    }
    __syncthreads();
}

// Link cache: the shared-memory image of phase A for every tile of both parities, built once per solve
// ([parity][tile] x sizeof(TileSmem<S>) bytes); dslash_tile_kernel<SL = 2> then stages a tile with ONE bulk copy
// (cp.async.bulk, the 1-D TMA path) instead of loading, converting and rebuilding the links in every launch.
template <int PREC, int RECON, int S>
__global__ void __launch_bounds__(256) link_cache_kernel(DslashKArgs a, char* cache, int tiles)
{
    __shared__ __align__(128) TileSmem<S> sm;
    a.parity = blockIdx.y;
    const int tile = blockIdx.x;
    // zero first: tail tiles leave unused slots, and the image is copied whole
    for (int i = threadIdx.x; i < (int)(sizeof(TileSmem<S>) / 4); i += blockDim.x) reinterpret_cast<int*>(&sm)[i] = 0;
    __syncthreads();
    tile_build<PREC, RECON, S>(a, tile * S, threadIdx.x, blockDim.x, sm);
    uint4* dst = reinterpret_cast<uint4*>(cache + ((size_t)blockIdx.y * tiles + tile) * sizeof(TileSmem<S>));
    for (int i = threadIdx.x; i < (int)(sizeof(TileSmem<S>) / 16); i += blockDim.x) dst[i] = reinterpret_cast<const uint4*>(&sm)[i];
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// SL: 0 = links loaded by each thread (nrhs = 1), 1 = tile links built into shared memory in the kernel
template <int PREC, int RECON, int DAG, int S, int RB, int MINB, int SL>
__global__ void __launch_bounds__(S* RB, MINB) dslash_tile_kernel(const DslashKArgs a)
{
    __shared__ __align__(128) TileSmem<SL ? S : 1> sm;

    const int tx = threadIdx.x, ty = threadIdx.y;
    const int ny = (a.nrhs + RB - 1) / RB;
    const int tile = blockIdx.x / ny, by = blockIdx.x - tile * ny; // rhs groups of one tile are adjacent in launch order
    const int cb0 = tile * S, cb = cb0 + tx, Vh = a.g.Vh;
    const int rhs = by * RB + ty;
    const bool valid = cb < Vh;
    const bool act = valid && rhs < a.nrhs && (a.active == nullptr || a.active[rhs] != 0);

    int nb[8];
    if constexpr (SL == 1) {
        if (__syncthreads_or(act) == 0) return;
        tile_build<PREC, RECON, S>(a, cb0, ty * S + tx, S * RB, sm);
    }
    if constexpr (SL != 0) {
        if (!act) return;
#pragma unroll
        for (int d = 0; d < 8; ++d) {
            const int v = sm.nbr[d][tx];
            nb[d] = (d >= 6 && v < 0) ? ~v : v;
        }
    }
    float sgp = 1.f, sgm = 1.f;
    if constexpr (!SL) {
        if (!act) return;
        tile_neighbours(a.g, a.parity, cb, nb, sgp, sgm);
#ifdef TM_DEBUG_L1WIN // timing ablation (probe builds only, wrong results): every gather lands inside the CTA's own site range
#pragma unroll
        for (int d = 0; d < 8; ++d) nb[d] = min(cb0 + (nb[d] & (S - 1)), Vh - 1);
#endif
    }

    tile_site_any<PREC, RECON, DAG, SL>(a, sm, cb, tx, rhs, nb, sgp, sgm);
}

// ---- multi-rhs kernel fed from the link cache ------------------------------------------------------------------
// A CTA walks TPC consecutive tiles.  The tile images (19 KB: neighbour indices + fp32 links) arrive by bulk copy
// (cp.async.bulk = 1-D TMA, completion on an mbarrier) into a two-deep ring, so the copy of tile i+1 overlaps the
// arithmetic of tile i and no thread spends an instruction on link addressing, conversion or reconstruction.
__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
    // the tile images are read once per launch: evict-first in L2, so that they do not push out the spinors being gathered
    const unsigned long long pol = link_policy();
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar), "l"(pol)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile("{\n\t.reg .pred p;\n\tTM_WAIT_%=:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t@p bra TM_DONE_%=;\n\tbra TM_WAIT_%=;\n\tTM_DONE_%=:\n\t}" ::"r"(bar),
                 "r"(parity)
                 : "memory");
}

template <int PREC, int RECON, int DAG, int RB, int MINB, int TPC>
__global__ void __launch_bounds__(32 * RB, MINB) dslash_tile_lc_kernel(const DslashKArgs a)
{
    constexpr int S = 32;
    constexpr uint32_t BYTES = (uint32_t)sizeof(TileSmem<S>);
    __shared__ __align__(128) TileSmem<S> sm[2];
    __shared__ __align__(8) unsigned long long bar[2];

    const int tx = threadIdx.x, ty = threadIdx.y;
    const int ny = (a.nrhs + RB - 1) / RB;
    const int grp = blockIdx.x / ny, by = blockIdx.x - grp * ny;
    const int Vh = a.g.Vh, tiles = (Vh + S - 1) / S;
    const int tile0 = grp * TPC;
    const int ntile = min(TPC, tiles - tile0);
    const int rhs = by * RB + ty;
    const bool ract = rhs < a.nrhs && (a.active == nullptr || a.active[rhs] != 0);
    const bool leader = (tx == 0 && ty == 0);
    const char* img = a.link_cache + ((size_t)a.parity * tiles + tile0) * sizeof(TileSmem<S>);
#ifdef TM_DEBUG_IMGWIN
    // timing ablation (probe builds only, wrong results): the LINKS of every tile image come from a 64-tile window of the cache (L2
    // hits, no DRAM traffic), the neighbour indices from the tile's own image (the gathers keep their addresses): two copies per image
    constexpr uint32_t NBYTES = (uint32_t)sizeof(((TileSmem<S>*)nullptr)->nbr);
    const char* imgw = a.link_cache + ((size_t)a.parity * tiles + (tile0 & 63)) * sizeof(TileSmem<S>);
#define TM_IMG_LOAD(buf, k)                                                                                              \
    do {                                                                                                                 \
        bulk_load(smem_u32(&sm[buf]), img + (size_t)(k) * sizeof(TileSmem<S>), NBYTES, smem_u32(&bar[buf]));             \
        bulk_load(smem_u32(&sm[buf]) + NBYTES, imgw + (size_t)((k) & 3) * sizeof(TileSmem<S>) + NBYTES, BYTES - NBYTES, smem_u32(&bar[buf])); \
    } while (0)
    constexpr int ARRIVALS = 2;
#else
#define TM_IMG_LOAD(buf, k) bulk_load(smem_u32(&sm[buf]), img + (size_t)(k) * sizeof(TileSmem<S>), BYTES, smem_u32(&bar[buf]))
    constexpr int ARRIVALS = 1;
#endif
    if (leader) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(&bar[0])), "r"(ARRIVALS) : "memory");
        asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(&bar[1])), "r"(ARRIVALS) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (__syncthreads_or(ract) == 0) return;
    if (leader) TM_IMG_LOAD(0, 0);
    // (decoupling the warps with per-buffer "empty" mbarriers instead of the CTA barrier was measured 2 % slower; two to six
    // right-hand sides per thread with the links kept in registers 15 % to 4.8 x slower: profiles/r02_ablations_12rhs_dslash.md)
    for (int i = 0; i < ntile; ++i) {
        const int b = i & 1;
        if (leader && i + 1 < ntile) // buffer b^1 was released by the barrier that closed tile i-1
            TM_IMG_LOAD(b ^ 1, i + 1);
        const int cb = (tile0 + i) * S + tx;
        if (ract && cb < Vh) {
            mbar_wait(smem_u32(&bar[b]), (i >> 1) & 1);
            int nb[8];
#pragma unroll
            for (int d = 0; d < 8; ++d) {
                const int v = sm[b].nbr[d][tx];
                nb[d] = (d >= 6 && v < 0) ? ~v : v; // only temporal hops carry the antiperiodic sign on their index
            }
            tile_site_any<PREC, RECON, DAG, 1>(a, sm[b], cb, tx, rhs, nb, 1.f, 1.f);
        }
        if (i + 1 < ntile) __syncthreads();
    }
}

#undef TM_IMG_LOAD

template <int PREC, int RECON, int RB, int MINB, int TPC>
static inline void launch_tile_lc(const DslashKArgs& a, bool dagger, cudaStream_t st)
{
    const int ny = (a.nrhs + RB - 1) / RB;
    const unsigned tiles = (unsigned)((a.g.Vh + 31) / 32);
    dim3 block(32, RB), grid(((tiles + TPC - 1) / TPC) * ny);
    if (dagger) dslash_tile_lc_kernel<PREC, RECON, 1, RB, MINB, TPC><<<grid, block, 0, st>>>(a);
    else dslash_tile_lc_kernel<PREC, RECON, 0, RB, MINB, TPC><<<grid, block, 0, st>>>(a);
}

template <int PREC, int RECON, int S, int RB, int MINB, int SL>
static inline void launch_tile(const DslashKArgs& a, bool dagger, cudaStream_t st)
{
    const int ny = (a.nrhs + RB - 1) / RB;
    const unsigned tiles = (unsigned)((a.g.Vh + S - 1) / S);
    dim3 block(S, RB), grid(tiles * ny);
    if (dagger) dslash_tile_kernel<PREC, RECON, 1, S, RB, MINB, SL><<<grid, block, 0, st>>>(a);
    else dslash_tile_kernel<PREC, RECON, 0, S, RB, MINB, SL><<<grid, block, 0, st>>>(a);
}

template <int PREC, int RECON>
static inline void launch_link_cache(const DslashKArgs& a, char* cache, cudaStream_t st)
{
    const int tiles = (a.g.Vh + 31) / 32;
    link_cache_kernel<PREC, RECON, 32><<<dim3(tiles, 2), 256, 0, st>>>(a, cache, tiles);
}

} // namespace tmk
