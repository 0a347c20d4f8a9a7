// tm_contract.cuh -- per-site colour-traced contraction of two raw fp16-storage spinors (shared by the time-slice loop kernel,
// tm_loop.cu, and the momentum-projected loops, tm_insert.cu; "Traces were taken in color space").
#pragma once
#include "tm_layout.cuh"

namespace tmk {

// fp16 storage: f32 += f16 * f16 (SASS FHFMA; the product of two binary16 numbers is exact in fp32), so the stored words are
// multiplied without conversion or norm scaling and the site's 32 sums are scaled once by norm_a * norm_b.
// HA / HB select the low (re) or high (im) half of the packed words, NEG negates the product.
template <int HA, int HB, int NEG>
__device__ __forceinline__ float fhfma(uint32_t wa, uint32_t wb, float c)
{
    float r;
#define TM_FHFMA(A, B, N) \
    asm("{.reg .b16 al,ah,bl,bh; mov.b32 {al,ah}, %1; mov.b32 {bl,bh}, %2; " N " fma.rn.f32.f16 %0, " A ", " B ", %3;}" : "=f"(r) : "r"(wa), "r"(wb), "f"(c))
    if (HA == 0 && HB == 0 && !NEG) TM_FHFMA("al", "bl", "");
    if (HA == 0 && HB == 1 && !NEG) TM_FHFMA("al", "bh", "");
    if (HA == 1 && HB == 0 && !NEG) TM_FHFMA("ah", "bl", "");
    if (HA == 1 && HB == 1 && !NEG) TM_FHFMA("ah", "bh", "");
    if (HA == 0 && HB == 0 && NEG) TM_FHFMA("al", "bl", "neg.f16 al, al;");
    if (HA == 0 && HB == 1 && NEG) TM_FHFMA("al", "bh", "neg.f16 al, al;");
    if (HA == 1 && HB == 0 && NEG) TM_FHFMA("ah", "bl", "neg.f16 ah, ah;");
    if (HA == 1 && HB == 1 && NEG) TM_FHFMA("ah", "bh", "neg.f16 ah, ah;");
#undef TM_FHFMA
    return r;
}
__device__ __forceinline__ uint32_t word_of(const uint4* q, int j) // complex number j = spin * 3 + colour of a raw fp16 site
{
    const uint4 v = q[j >> 2];
    return (j & 3) == 0 ? v.x : (j & 3) == 1 ? v.y : (j & 3) == 2 ? v.z : v.w;
}
// accf[32] += norm_a norm_b * sum_c conj(a_{al c}) b_{be c} from the raw words of one site
__device__ __forceinline__ void site_contract_h(const uint4* qa, float na, const uint4* qb, float nb_, float* accf)
{
    const float w = na * nb_;
#pragma unroll
    for (int al = 0; al < 4; ++al)
#pragma unroll
        for (int be = 0; be < 4; ++be) {
            float re = 0.f, im = 0.f;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const uint32_t wa = word_of(qa, al * 3 + c), wb = word_of(qb, be * 3 + c);
                re = fhfma<0, 0, 0>(wa, wb, re); // ar br
                re = fhfma<1, 1, 0>(wa, wb, re); // ai bi
                im = fhfma<0, 1, 0>(wa, wb, im); // ar bi
                im = fhfma<1, 0, 1>(wa, wb, im); // -ai br
            }
            accf[(al * 4 + be) * 2] = fmaf(w, re, accf[(al * 4 + be) * 2]);
            accf[(al * 4 + be) * 2 + 1] = fmaf(w, im, accf[(al * 4 + be) * 2 + 1]);
        }
}

} // namespace tmk
