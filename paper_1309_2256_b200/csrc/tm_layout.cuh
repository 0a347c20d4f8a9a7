// tm_layout.cuh -- packed device layout: even-odd structure of arrays in 16-byte chunks.
//
// One-parity spinor, Vh sites, checkerboard index cb:
//   real r = (spin*3 + colour)*2 + reim, r = 0..23
//   fp64: 12 chunks of double2  -> chunk k holds reals 2k, 2k+1       at ((double2*)base)[k*Vh + cb]
//   fp32:  6 chunks of float4   -> chunk k holds reals 4k..4k+3       at ((float4*)base)[k*Vh + cb]
//   fp16:  3 chunks of 8 halves -> chunk k holds reals 8k..8k+7       at ((uint4*)base)[k*Vh + cb]
//          followed by Vh fp32 norms; value = half * norm, norm = max |real| of the site (north_star:
//          "fp16 storage with a per-site fp32 norm").
// One (parity, mu) link block, R = 18 or 12 reals per link, real r = (row*3 + col)*2 + reim:
//   fp64: R/2 chunks of double2
//   fp32: 18 -> 4 float4 chunks + 1 float2 tail array; 12 -> 3 float4 chunks
//   fp16: 18 -> 2 uint4 chunks + 1 half2 (4-byte) tail array; 12 -> 1 uint4 chunk + 1 uint2 (8-byte) tail array
// Links are stored unscaled (|U_ij| <= 1).  With R = 12 the third row is rebuilt as conj(row0 x row1)
// ("12-parameter reconstruction").  R = 8 ("8-parameter reconstruction ... only the coefficients
// are stored (8 real numbers)"; the paper gives no formulas, reading 31): U01, U02, U10 and the phases of U00 and U20
// in units of pi; fp64: 4 double2 chunks, fp32: 2 float4, fp16: 1 uint4.  rebuild_from8() below.
#pragma once
#include "tm_common.cuh"

namespace tmk {

template <int PREC> struct Prec;
template <> struct Prec<8> { typedef double real; };
template <> struct Prec<4> { typedef float real; };
template <> struct Prec<2> { typedef float real; };

__device__ __forceinline__ uint4 ldg128(const void* p) { return __ldg(reinterpret_cast<const uint4*>(p)); }
__device__ __forceinline__ uint2 ldg64(const void* p) { return __ldg(reinterpret_cast<const uint2*>(p)); }
__device__ __forceinline__ uint32_t ldg32(const void* p) { return __ldg(reinterpret_cast<const uint32_t*>(p)); }

// Link loads: every link is read exactly once per launch, so it is fetched with an L2 evict-first policy and without L1
// allocation -- the neighbour spinors (each gathered by eight sites) keep the L2 (matters once the lattice outgrows it).
#ifndef TM_LINK_STREAM
#define TM_LINK_STREAM 1
#endif
__device__ __forceinline__ unsigned long long link_policy()
{
    unsigned long long pol;
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// Same hints on a COHERENT load (no .nc): for an operand that the same kernel also writes -- the y of a fused axpy may be the
// output vector itself (r = r - alpha A p), and the non-coherent path requires data that is read-only for the whole kernel.
template <typename T>
__device__ __forceinline__ T stream_ld(const T* p)
{
    const unsigned long long pol = link_policy();
    T v;
    if constexpr (sizeof(T) == 16) {
        uint4 q;
        asm volatile("ld.global.L1::no_allocate.L2::cache_hint.v4.u32 {%0,%1,%2,%3}, [%4], %5;" : "=r"(q.x), "=r"(q.y), "=r"(q.z), "=r"(q.w) : "l"(p), "l"(pol) : "memory");
        v = *reinterpret_cast<const T*>(&q);
    } else if constexpr (sizeof(T) == 8) {
        uint2 q;
        asm volatile("ld.global.L1::no_allocate.L2::cache_hint.v2.u32 {%0,%1}, [%2], %3;" : "=r"(q.x), "=r"(q.y) : "l"(p), "l"(pol) : "memory");
        v = *reinterpret_cast<const T*>(&q);
    } else {
        uint32_t q;
        asm volatile("ld.global.L1::no_allocate.L2::cache_hint.u32 %0, [%1], %2;" : "=r"(q) : "l"(p), "l"(pol) : "memory");
        v = *reinterpret_cast<const T*>(&q);
    }
    return v;
}

template <typename T>
__device__ __forceinline__ T link_ldg(const T* p)
{
#if TM_LINK_STREAM
    const unsigned long long pol = link_policy();
    T v;
    if constexpr (sizeof(T) == 16) {
        uint4 q;
        asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.u32 {%0,%1,%2,%3}, [%4], %5;" : "=r"(q.x), "=r"(q.y), "=r"(q.z), "=r"(q.w) : "l"(p), "l"(pol));
        v = *reinterpret_cast<const T*>(&q);
    } else if constexpr (sizeof(T) == 8) {
        uint2 q;
        asm("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.u32 {%0,%1}, [%2], %3;" : "=r"(q.x), "=r"(q.y) : "l"(p), "l"(pol));
        v = *reinterpret_cast<const T*>(&q);
    } else {
        uint32_t q;
        asm("ld.global.nc.L1::no_allocate.L2::cache_hint.u32 %0, [%1], %2;" : "=r"(q) : "l"(p), "l"(pol));
        v = *reinterpret_cast<const T*>(&q);
    }
    return v;
#else
    return __ldg(p);
#endif
}

__device__ __forceinline__ void unpack_h2(uint32_t w, float& a, float& b)
{
    const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&w));
    a = f.x;
    b = f.y;
}
__device__ __forceinline__ uint32_t pack_h2(float a, float b)
{
    const __half2 h = __floats2half2_rn(a, b);
    return *reinterpret_cast<const uint32_t*>(&h);
}

// 16-bit fixed-point link words (TM_RECON_*_FIX16, tm.h): each half of w is the offset-binary word q + 32768 of a real q / 32767.
// 0x4B000000 | word is the float 2^23 + word exactly, so one byte permute, one exact subtraction and one multiply convert
// it on the FMA / ALU pipes (an I2F per real would queue on the quarter-rate conversion unit).
__device__ __forceinline__ void unpack_q2(uint32_t w, float& a, float& b)
{
    const float fa = __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7610));
    const float fb = __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7632));
    a = (fa - 8421376.0f) * (1.0f / 32767.0f);
    b = (fb - 8421376.0f) * (1.0f / 32767.0f);
}
template <bool FX>
__device__ __forceinline__ void unpack_w2(uint32_t w, float& a, float& b)
{
    if constexpr (FX) unpack_q2(w, a, b);
    else unpack_h2(w, a, b);
}

// ------------------------------------------------------------------------------------------------
// spinor load: v[24] in arithmetic precision
// ------------------------------------------------------------------------------------------------
// STREAM 1: the operand is read exactly once per launch and never written by it (the x of an XPAY epilogue): evict-first, non-coherent
// like the links.  STREAM 2: read once but possibly ALIASED by the kernel's output (the y of a fused axpy): same hints, coherent load.
template <int PREC, int STREAM = 0>
__device__ __forceinline__ void load_spinor(const void* base, int Vh, int cb, typename Prec<PREC>::real* v)
{
    if constexpr (PREC == 8) {
        const double2* p = reinterpret_cast<const double2*>(base) + cb;
#pragma unroll
        for (int k = 0; k < 12; ++k) {
            const double2 d = STREAM == 2 ? stream_ld(p + (size_t)k * Vh) : STREAM == 1 ? link_ldg(p + (size_t)k * Vh) : __ldg(p + (size_t)k * Vh);
            v[2 * k] = d.x;
            v[2 * k + 1] = d.y;
        }
    } else if constexpr (PREC == 4) {
        const float4* p = reinterpret_cast<const float4*>(base) + cb;
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            const float4 d = STREAM == 2 ? stream_ld(p + (size_t)k * Vh) : STREAM == 1 ? link_ldg(p + (size_t)k * Vh) : __ldg(p + (size_t)k * Vh);
            v[4 * k] = d.x;
            v[4 * k + 1] = d.y;
            v[4 * k + 2] = d.z;
            v[4 * k + 3] = d.w;
        }
    } else {
        const uint4* p = reinterpret_cast<const uint4*>(base) + cb;
        uint4 q[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) q[k] = STREAM == 2 ? stream_ld(p + (size_t)k * Vh) : STREAM == 1 ? link_ldg(p + (size_t)k * Vh) : __ldg(p + (size_t)k * Vh);
        const float* np_ = reinterpret_cast<const float*>(reinterpret_cast<const uint4*>(base) + (size_t)3 * Vh) + cb;
        const float nrm = STREAM == 2 ? stream_ld(np_) : STREAM == 1 ? link_ldg(np_) : __ldg(np_);
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            unpack_h2(q[k].x, v[8 * k + 0], v[8 * k + 1]);
            unpack_h2(q[k].y, v[8 * k + 2], v[8 * k + 3]);
            unpack_h2(q[k].z, v[8 * k + 4], v[8 * k + 5]);
            unpack_h2(q[k].w, v[8 * k + 6], v[8 * k + 7]);
        }
#pragma unroll
        for (int r = 0; r < 24; ++r) v[r] *= nrm;
    }
}

template <int PREC>
__device__ __forceinline__ void store_spinor(void* base, int Vh, int cb, const typename Prec<PREC>::real* v)
{
    if constexpr (PREC == 8) {
        double2* p = reinterpret_cast<double2*>(base) + cb;
#pragma unroll
        for (int k = 0; k < 12; ++k) p[(size_t)k * Vh] = make_double2(v[2 * k], v[2 * k + 1]);
    } else if constexpr (PREC == 4) {
        float4* p = reinterpret_cast<float4*>(base) + cb;
#pragma unroll
        for (int k = 0; k < 6; ++k) p[(size_t)k * Vh] = make_float4(v[4 * k], v[4 * k + 1], v[4 * k + 2], v[4 * k + 3]);
    } else {
        float m = 0.f;
#pragma unroll
        for (int r = 0; r < 24; ++r) m = fmaxf(m, fabsf(v[r]));
        const float inv = (m > 0.f) ? __fdividef(1.0f, m) : 0.f;
        uint4* p = reinterpret_cast<uint4*>(base) + cb;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            uint4 q;
            q.x = pack_h2(v[8 * k + 0] * inv, v[8 * k + 1] * inv);
            q.y = pack_h2(v[8 * k + 2] * inv, v[8 * k + 3] * inv);
            q.z = pack_h2(v[8 * k + 4] * inv, v[8 * k + 5] * inv);
            q.w = pack_h2(v[8 * k + 6] * inv, v[8 * k + 7] * inv);
            p[(size_t)k * Vh] = q;
        }
        reinterpret_cast<float*>(reinterpret_cast<uint4*>(base) + (size_t)3 * Vh)[cb] = m;
    }
}

// ------------------------------------------------------------------------------------------------
// link load: u[18] (row-major complex 3x3); RECON 12 rebuilds row 2
// ------------------------------------------------------------------------------------------------
template <typename real>
__device__ __forceinline__ void rebuild_row2(real* u)
{
    // row2_j = conj(row0_{j+1} row1_{j+2} - row0_{j+2} row1_{j+1})
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const int j1 = (j + 1) % 3, j2 = (j + 2) % 3;
        const real ar = u[2 * j1], ai = u[2 * j1 + 1], br = u[6 + 2 * j2], bi = u[6 + 2 * j2 + 1];
        const real cr = u[2 * j2], ci = u[2 * j2 + 1], dr = u[6 + 2 * j1], di = u[6 + 2 * j1 + 1];
        // one multiply + three FMAs per real (8 instead of 10 operations per complex entry)
        u[12 + 2 * j] = fma(ci, di, fma(-cr, dr, fma(-ai, bi, ar * br)));
        u[12 + 2 * j + 1] = fma(ci, dr, fma(cr, di, fma(-ai, br, -(ar * bi))));
    }
}

// 8 stored reals q = (V01, V02, V10, arg V00 / pi, arg V20 / pi) of V = U P, V_ij = U_{i,(j+2)%3} (a cyclic column shift: det P = 1, so V
// is in SU(3); it moves the chart's singular set V01 = V02 = 0 from the unit link -- which every free field and every temporal-gauge
// field is full of -- to |U02| = 1) -> u[18].  Unitarity of row 0 and column 0 gives |U00|, |U20|;
// row 1 follows from  row1 . conj(row0) = 0  and  (row0 x row1)_0 = conj(U20)  (two linear equations in U11, U12 with determinant
// r = |U01|^2 + |U02|^2), row 2 = conj(row0 x row1).  Ill-conditioned as r -> 0 (errors grow like 1/r).
template <typename real>
__device__ __forceinline__ void rebuild_from8(const real* q, real* u)
{
    const real a1r = q[0], a1i = q[1], a2r = q[2], a2i = q[3], br = q[4], bi = q[5];
    const real r = a1r * a1r + a1i * a1i + a2r * a2r + a2i * a2i;
    const real m00 = sqrt(fmax(real(0), real(1) - r));
    real s0, c0, s1, c1;
    sincospi(q[6], &s0, &c0);
    sincospi(q[7], &s1, &c1);
    const real u00r = m00 * c0, u00i = m00 * s0;
    const real m20 = sqrt(fmax(real(0), r - br * br - bi * bi));
    const real u20r = m20 * c1, u20i = m20 * s1;
    const real rinv = real(1) / r;
    // t = U10 conj(U00)
    const real tr = br * u00r + bi * u00i, ti = bi * u00r - br * u00i;
    // U11 = -(t U01 + conj(U02) conj(U20)) / r ; conj(U02) conj(U20) = conj(U02 U20)
    const real pr = a2r * u20r - a2i * u20i, pi_ = a2r * u20i + a2i * u20r; // U02 U20
    const real u11r = -(tr * a1r - ti * a1i + pr) * rinv, u11i = -(tr * a1i + ti * a1r - pi_) * rinv;
    // U12 = (conj(U01 U20) - t U02) / r
    const real wr = a1r * u20r - a1i * u20i, wi = a1r * u20i + a1i * u20r; // U01 U20
    const real u12r = (wr - (tr * a2r - ti * a2i)) * rinv, u12i = (-wi - (tr * a2i + ti * a2r)) * rinv;
    real v[18]; // the stored matrix is V = U P (columns shifted cyclically, below)
    v[0] = u00r; v[1] = u00i; v[2] = a1r; v[3] = a1i; v[4] = a2r; v[5] = a2i;
    v[6] = br; v[7] = bi; v[8] = u11r; v[9] = u11i; v[10] = u12r; v[11] = u12i;
    rebuild_row2(v);
    // U_{i,(j+2)%3} = V_{ij}: undoing the column shift is a renaming of registers
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            u[2 * (i * 3 + (j + 2) % 3)] = v[2 * (i * 3 + j)];
            u[2 * (i * 3 + (j + 2) % 3) + 1] = v[2 * (i * 3 + j) + 1];
        }
}

template <int PREC, int RECON_CODE>
__device__ __forceinline__ void load_link(const void* block, int Vh, int cb, typename Prec<PREC>::real* u)
{
    constexpr int RECON = RECON_CODE % 100;                  // reals stored per link
    constexpr bool FX = (RECON_CODE / 100 == 1) && (PREC == 2); // 16-bit words are fixed point instead of binary16
    static_assert(RECON_CODE < 100 || RECON == 18 || RECON == 12, "fixed-point / temporal-gauge codes: 18 or 12 reals");
    if constexpr (RECON == 8) {
        typename Prec<PREC>::real q[8];
        if constexpr (PREC == 8) {
            const double2* p = reinterpret_cast<const double2*>(block) + cb;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const double2 d = link_ldg(p + (size_t)k * Vh);
                q[2 * k] = d.x;
                q[2 * k + 1] = d.y;
            }
        } else if constexpr (PREC == 4) {
            const float4* p = reinterpret_cast<const float4*>(block) + cb;
            const float4 d0 = link_ldg(p), d1 = link_ldg(p + (size_t)Vh);
            q[0] = d0.x; q[1] = d0.y; q[2] = d0.z; q[3] = d0.w;
            q[4] = d1.x; q[5] = d1.y; q[6] = d1.z; q[7] = d1.w;
        } else {
            const uint4 d = link_ldg(reinterpret_cast<const uint4*>(block) + cb);
            unpack_h2(d.x, q[0], q[1]);
            unpack_h2(d.y, q[2], q[3]);
            unpack_h2(d.z, q[4], q[5]);
            unpack_h2(d.w, q[6], q[7]);
        }
        rebuild_from8(q, u);
        return;
    } else if constexpr (PREC == 8) {
        const double2* p = reinterpret_cast<const double2*>(block) + cb;
#pragma unroll
        for (int k = 0; k < RECON / 2; ++k) {
            const double2 d = link_ldg(p + (size_t)k * Vh);
            u[2 * k] = d.x;
            u[2 * k + 1] = d.y;
        }
    } else if constexpr (PREC == 4) {
        const float4* p = reinterpret_cast<const float4*>(block) + cb;
#pragma unroll
        for (int k = 0; k < RECON / 4; ++k) {
            const float4 d = link_ldg(p + (size_t)k * Vh);
            u[4 * k] = d.x;
            u[4 * k + 1] = d.y;
            u[4 * k + 2] = d.z;
            u[4 * k + 3] = d.w;
        }
        if constexpr (RECON == 18) {
            const float2 d = link_ldg(reinterpret_cast<const float2*>(reinterpret_cast<const float4*>(block) + (size_t)4 * Vh) + cb);
            u[16] = d.x;
            u[17] = d.y;
        }
    } else {
        const uint4* p = reinterpret_cast<const uint4*>(block) + cb;
        constexpr int NC = RECON / 8; // 2 or 1 full chunks
#pragma unroll
        for (int k = 0; k < NC; ++k) {
            const uint4 q = link_ldg(p + (size_t)k * Vh);
            unpack_w2<FX>(q.x, u[8 * k + 0], u[8 * k + 1]);
            unpack_w2<FX>(q.y, u[8 * k + 2], u[8 * k + 3]);
            unpack_w2<FX>(q.z, u[8 * k + 4], u[8 * k + 5]);
            unpack_w2<FX>(q.w, u[8 * k + 6], u[8 * k + 7]);
        }
        const void* tail = reinterpret_cast<const uint4*>(block) + (size_t)NC * Vh;
        if constexpr (RECON == 18) {
            unpack_w2<FX>(link_ldg(reinterpret_cast<const uint32_t*>(tail) + cb), u[16], u[17]);
        } else {
            const uint2 q = link_ldg(reinterpret_cast<const uint2*>(tail) + cb);
            unpack_w2<FX>(q.x, u[8], u[9]);
            unpack_w2<FX>(q.y, u[10], u[11]);
        }
    }
#ifdef TM_DEBUG_NOREBUILD // timing ablation (probe builds only, wrong results): the third row is not rebuilt
    if constexpr (RECON == 12) {
#pragma unroll
        for (int k = 0; k < 6; ++k) u[12 + k] = u[k];
    }
#else
    if constexpr (RECON == 12) rebuild_row2(u);
#endif
}

} // namespace tmk
