// tm_estimators.cu -- SURVEY.md 8(f) NEXT-1: what turns the kernels into the paper's estimators.
//
//   tm_M            full operator M(kappa,mu) psi = R psi - kappa Dslash psi on both parities (two fused dslash launches);
//                   mu = 0 gives the Wilson operator D_W = (M_u + M_d)/2 of Eq. (14).
//   tm_oneend_loops one-end trick loops from a solution s = M(kappa,+mu)^-1 eta:
//                   TAU3     out = 2i a  sum_x s^dag g5 Gamma_n s,          a = 2 kappa mu        (Eq. 13)
//                   GENERAL  out = 2     sum_x s^dag g5 Gamma_n g5 D_W s                          (Eq. 15)
//                   With s = M_u^-1 eta the noise average of TAU3 is Tr(M_d^-1 X) - Tr(M_u^-1 X) (reading 25:
//                   the sign of Eq. 13 as printed holds for s = M_d^-1 eta) and of GENERAL Tr(M_u^-1 X) + Tr(M_d^-1 X).
//   tm_tsm_combine  Eq. (8): L = 1/N_HP sum_r [L_HP(r) - L_LP(r)] + 1/N_LP sum_j L_LP(j)
#include "tm_common.cuh"

namespace tmk {

// out_full = (1 + i a g5) in - kappa Dslash in, a = +-2 kappa mu (sign - and projector signs flipped if dagger)
int full_operator(const Geo& g, const void* gauge, int prec, int recon, void* out_full, const void* in_full, double kappa, double mu,
                  int dagger, int nrhs, cudaStream_t st)
{
    const size_t pb = spinor_parity_bytes(g, prec);
    const double a = 2.0 * kappa * mu * (dagger ? -1.0 : 1.0);
    DslashParams p;
    p.gauge = gauge; p.nrhs = nrhs; p.active = nullptr; p.dagger = dagger ? 1 : 0;
    p.rhs_stride_out = p.rhs_stride_in = p.rhs_stride_x = 2 * pb;
    p.pq[0] = 1.0; p.pq[1] = a; p.pq[2] = -kappa; p.pq[3] = 0.0;
    for (int parity = 0; parity < 2; ++parity) {
        p.out = static_cast<char*>(out_full) + parity * pb;
        p.in = static_cast<const char*>(in_full) + (1 - parity) * pb;
        p.x = static_cast<const char*>(in_full) + parity * pb;
        p.out_parity = parity;
        const int rc = launch_dslash(g, prec, recon, p, st);
        if (rc != TM_OK) return rc;
    }
    return TM_OK;
}

// out[n][t] = 1/nhp sum_r (hp[r] - lpc[r]) + 1/nlp sum_j lp[j], fixed summation order; one thread per real of [16][T][2]
__global__ void tsm_combine_kernel(int n, const double* hp, const double* lpc, int nhp, const double* lp, int nlp, double* out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double c = 0.0, l = 0.0;
    for (int r = 0; r < nhp; ++r) c += hp[(size_t)r * n + i] - lpc[(size_t)r * n + i];
    for (int j = 0; j < nlp; ++j) l += lp[(size_t)j * n + i];
    out[i] = (nhp > 0 ? c / nhp : 0.0) + (nlp > 0 ? l / nlp : 0.0);
}

} // namespace tmk

using namespace tmk;

extern "C" int tm_M(const tm_lattice* L, const void* gauge, int prec, int recon, void* out_full, const void* in_full, double kappa,
                    double mu, int dagger, int nrhs, void* stream)
{
    if (!L || !gauge || !out_full || !in_full || !valid_prec(prec) || !valid_recon(recon)) return TM_ERR_ARG;
    if (out_full == in_full || nrhs < 1 || nrhs > TM_MAX_NRHS) return TM_ERR_ARG;
    if (!aligned256(gauge) || !aligned256(out_full) || !aligned256(in_full)) return TM_ERR_LAYOUT;
    return full_operator(L->g, gauge, prec, recon, out_full, in_full, kappa, mu, dagger, nrhs, (cudaStream_t)stream);
}

extern "C" size_t tm_oneend_workspace_bytes(const tm_lattice* L, int prec, int nrhs)
{
    if (!L || !valid_prec(prec) || nrhs < 1) return 0;
    return round256(2 * spinor_parity_bytes(L->g, prec) * (size_t)nrhs) + loop_workspace_bytes(L->g, nrhs);
}

extern "C" int tm_oneend_loops(const tm_lattice* L, const void* gauge, int prec, int recon, const void* s_full, int kind, double kappa,
                               double mu, int nrhs, double* out, void* workspace, size_t workspace_bytes, void* stream)
{
    if (!L || !s_full || !out || !workspace || !valid_prec(prec) || nrhs < 1 || nrhs > TM_MAX_NRHS) return TM_ERR_ARG;
    if (kind != TM_ONEEND_TAU3 && kind != TM_ONEEND_GENERAL) return TM_ERR_ARG;
    if (!aligned256(s_full) || !aligned256(out) || !aligned256(workspace)) return TM_ERR_LAYOUT;
    if (workspace_bytes < tm_oneend_workspace_bytes(L, prec, nrhs)) return TM_ERR_LAYOUT;
    cudaStream_t st = (cudaStream_t)stream;
    char* w = static_cast<char*>(workspace);
    const size_t fb = round256(2 * spinor_parity_bytes(L->g, prec) * (size_t)nrhs);
    if (kind == TM_ONEEND_TAU3) // 2 i a (g5 s)^dag Gamma_n s
        return loop_contract_ex(L->g, s_full, s_full, prec, nrhs, out, w + fb, 1, 0, 0.0, 2.0 * (2.0 * kappa * mu), st);
    if (!gauge || !valid_recon(recon) || !aligned256(gauge)) return TM_ERR_ARG;
    // w = D_W s = M(kappa, 0) s ; out = 2 (g5 s)^dag Gamma_n (g5 w)
    const int rc = full_operator(L->g, gauge, prec, recon, w, s_full, kappa, 0.0, 0, nrhs, st);
    if (rc != TM_OK) return rc;
    return loop_contract_ex(L->g, s_full, w, prec, nrhs, out, w + fb, 1, 1, 2.0, 0.0, st);
}

extern "C" int tm_tsm_combine(int T, const double* loops_hp, const double* loops_lp_same, int n_hp, const double* loops_lp, int n_lp,
                              double* out, void* stream)
{
    if (T < 1 || !out || n_hp < 0 || n_lp < 0 || (n_hp > 0 && (!loops_hp || !loops_lp_same)) || (n_lp > 0 && !loops_lp))
        return TM_ERR_ARG;
    const int n = 16 * T * 2;
    tsm_combine_kernel<<<(n + 127) / 128, 128, 0, (cudaStream_t)stream>>>(n, loops_hp, loops_lp_same, n_hp, loops_lp, n_lp, out);
    TM_LAUNCH_CHECK("tsm_combine_kernel");
    return TM_OK;
}
