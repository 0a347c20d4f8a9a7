// tm_loop.cu -- a8 of SURVEY.md 8(a): per-time-slice stochastic loop contraction for the 16 Gamma_n.
//
//   L[n][t] = sum_{x: x4=t} a(x)^dag (Gamma_n x 1_colour) b(x)          (Eq. 10)
// computed as the colour-traced Dirac-open 4x4 matrix C_{al be}(t) = sum_x sum_c conj(a_{al c}) b_{be c}
// ("Traces were taken in color space, leaving the Dirac ... indices open ... a 4x4 matrix was
// obtained, with enough information to reconstruct any arbitrary gamma insertion") followed by
// L[n][t] = sum_{al be} (Gamma_n)_{al be} C_{al be}(t).
// Time slice t of parity p is the contiguous checkerboard range [t*V3h, (t+1)*V3h).
// Reduction: per-site products in the storage arithmetic (fp32 for fp32/fp16 inputs), summed in that arithmetic over
// at most LOOP_CHUNK = 8 sites of a thread, then fp64: per-thread accumulator, warp shuffles, shared memory across warps, per-block partials, then one fixed-order final pass:
// bit-reproducible, no floating-point atomics.
#include "tm_layout.cuh"
#include "tm_gamma.cuh"
#include "tm_contract.cuh"
#include <mutex>

namespace tmk {

constexpr int LOOP_THREADS = 128;
constexpr int LOOP_CHUNK = 8; // sites summed in the storage arithmetic before the fp64 accumulator takes over

template <int PREC>
__global__ void __launch_bounds__(LOOP_THREADS, PREC == 2 ? 5 : 1) loop_partial_kernel(Geo g, const char* a_full, const char* b_full,
                                                                    size_t parity_bytes, double* partial, int nb, int t0)
{
    typedef typename Prec<PREC>::real real;
    const int t = t0 + blockIdx.y, rhs = blockIdx.z; // gridDim.y time slices starting at t0

    const char* af = a_full + (size_t)rhs * 2 * parity_bytes;
    const char* bf = b_full + (size_t)rhs * 2 * parity_bytes;
    // per-thread partial sums: products and the sum over up to LOOP_CHUNK sites in the storage arithmetic, then fp64
    double acc[32];
    real accf[32];
#pragma unroll
    for (int k = 0; k < 32; ++k) {
        acc[k] = 0.0;
        accf[k] = 0;
    }
    const int nsite = 2 * g.V3h;
    int pending = 0;
    for (int i = blockIdx.x * LOOP_THREADS + threadIdx.x; i < nsite; i += nb * LOOP_THREADS) {
        const int parity = i >= g.V3h;
        const int cb = t * g.V3h + (i - parity * g.V3h);
        if constexpr (PREC == 2) {
            uint4 qa[3], qb[3];
            const uint4* pa = reinterpret_cast<const uint4*>(af + parity * parity_bytes) + cb;
            const uint4* pb = reinterpret_cast<const uint4*>(bf + parity * parity_bytes) + cb;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                qa[k] = __ldg(pa + (size_t)k * g.Vh);
                qb[k] = __ldg(pb + (size_t)k * g.Vh);
            }
            const float na = __ldg(reinterpret_cast<const float*>(reinterpret_cast<const uint4*>(af + parity * parity_bytes) + (size_t)3 * g.Vh) + cb);
            const float nb_ = __ldg(reinterpret_cast<const float*>(reinterpret_cast<const uint4*>(bf + parity * parity_bytes) + (size_t)3 * g.Vh) + cb);
            site_contract_h(qa, na, qb, nb_, accf);
        } else {
            real a[24], b[24];
            load_spinor<PREC>(af + parity * parity_bytes, g.Vh, cb, a);
            load_spinor<PREC>(bf + parity * parity_bytes, g.Vh, cb, b);
#pragma unroll
            for (int al = 0; al < 4; ++al)
#pragma unroll
                for (int be = 0; be < 4; ++be) {
                    real re = accf[(al * 4 + be) * 2], im = accf[(al * 4 + be) * 2 + 1];
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const real ar = a[(al * 3 + c) * 2], ai = a[(al * 3 + c) * 2 + 1];
                        const real br = b[(be * 3 + c) * 2], bi = b[(be * 3 + c) * 2 + 1];
                        re = fma(ar, br, re);
                        re = fma(ai, bi, re);
                        im = fma(ar, bi, im);
                        im = fma(-ai, br, im);
                    }
                    accf[(al * 4 + be) * 2] = re;
                    accf[(al * 4 + be) * 2 + 1] = im;
                }
        }
        if (++pending == LOOP_CHUNK) {
#pragma unroll
            for (int k = 0; k < 32; ++k) {
                acc[k] += (double)accf[k];
                accf[k] = 0;
            }
            pending = 0;
        }
    }
#pragma unroll
    for (int k = 0; k < 32; ++k) acc[k] += (double)accf[k];
    __shared__ double sm[LOOP_THREADS / 32][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < 32; ++k) {
        double v = acc[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (lane == 0) sm[warp][k] = v;
    }
    __syncthreads();
    if (threadIdx.x < 32) {
        double v = 0.0;
#pragma unroll
        for (int w = 0; w < LOOP_THREADS / 32; ++w) v += sm[w][threadIdx.x];
        partial[(((size_t)rhs * gridDim.y + blockIdx.y) * nb + blockIdx.x) * 32 + threadIdx.x] = v;
    }
}

// out = scale * sum_{al be} (Gamma_n)_{al be} s5(al)^g5_left s5(be)^g5_right C_{al be}(t), s5 = (1,1,-1,-1) = diag g5:
// the bilinear (g5^l a)^dag Gamma_n (g5^r b) of the one-end trick (PAPER.md:127 Eq. 13, :141 Eq. 15)
__global__ void loop_final_kernel(int T, int nb, const double* partial, GammaTable tb, double* out, int g5_left, int g5_right,
                                  double scale_re, double scale_im)
{
    const int t = blockIdx.x, rhs = blockIdx.y;
    __shared__ double C[32];
    if (threadIdx.x < 32) {
        double v = 0.0;
        const double* p = partial + ((size_t)rhs * T + t) * nb * 32 + threadIdx.x;
        for (int b = 0; b < nb; ++b) v += p[(size_t)b * 32];
        C[threadIdx.x] = v;
    }
    __syncthreads();
    if (threadIdx.x < 16) {
        const int n = threadIdx.x;
        double re = 0.0, im = 0.0;
#pragma unroll
        for (int al = 0; al < 4; ++al) {
            const int be = tb.col[n][al];
            const double gr = tb.re[n][al], gi = tb.im[n][al];
            const double sg = ((g5_left && al >= 2) ? -1.0 : 1.0) * ((g5_right && be >= 2) ? -1.0 : 1.0);
            const double cr = sg * C[(al * 4 + be) * 2], ci = sg * C[(al * 4 + be) * 2 + 1];
            re += gr * cr - gi * ci;
            im += gr * ci + gi * cr;
        }
        out[(((size_t)rhs * 16 + n) * T + t) * 2] = scale_re * re - scale_im * im;
        out[(((size_t)rhs * 16 + n) * T + t) * 2 + 1] = scale_re * im + scale_im * re;
    }
}

static int loop_nb(const Geo& g)
{
    int nb = (2 * g.V3h) / (LOOP_THREADS * 16);
    if (nb < 1) nb = 1;
    if (nb > 32) nb = 32;
    return nb;
}

// time slices [t0, t0 + nt): out[rhs][16][nt][2]
int loop_contract_range(const Geo& g, const void* a_full, const void* b_full, int prec, int nrhs, double* out, void* workspace,
                        int g5_left, int g5_right, double scale_re, double scale_im, int t0, int nt, cudaStream_t st)
{
    static const GammaTable tb = make_gamma_table();
    const int nb = loop_nb(g);
    dim3 grid(nb, nt, nrhs), block(LOOP_THREADS);
    const size_t pb = spinor_parity_bytes(g, prec);
    double* partial = static_cast<double*>(workspace);
    if (prec == 8) loop_partial_kernel<8><<<grid, block, 0, st>>>(g, (const char*)a_full, (const char*)b_full, pb, partial, nb, t0);
    else if (prec == 4) loop_partial_kernel<4><<<grid, block, 0, st>>>(g, (const char*)a_full, (const char*)b_full, pb, partial, nb, t0);
    else loop_partial_kernel<2><<<grid, block, 0, st>>>(g, (const char*)a_full, (const char*)b_full, pb, partial, nb, t0);
    TM_LAUNCH_CHECK("loop_partial_kernel");
    loop_final_kernel<<<dim3(nt, nrhs), 32, 0, st>>>(nt, nb, partial, tb, out, g5_left, g5_right, scale_re, scale_im);
    TM_LAUNCH_CHECK("loop_final_kernel");
    return TM_OK;
}

int loop_contract_ex(const Geo& g, const void* a_full, const void* b_full, int prec, int nrhs, double* out, void* workspace,
                     int g5_left, int g5_right, double scale_re, double scale_im, cudaStream_t st)
{
    return loop_contract_range(g, a_full, b_full, prec, nrhs, out, workspace, g5_left, g5_right, scale_re, scale_im, 0, g.T, st);
}

int loop_contract(const Geo& g, const void* a_full, const void* b_full, int prec, int nrhs, double* out, void* workspace,
                  cudaStream_t st)
{
    return loop_contract_ex(g, a_full, b_full, prec, nrhs, out, workspace, 0, 0, 1.0, 0.0, st);
}

size_t loop_workspace_bytes(const Geo& g, int nrhs) { return round256((size_t)nrhs * g.T * loop_nb(g) * 32 * sizeof(double)); }

} // namespace tmk

using namespace tmk;

extern "C" size_t tm_loop_workspace_bytes(const tm_lattice* L, int nrhs)
{
    if (!L || nrhs < 1) return 0;
    return loop_workspace_bytes(L->g, nrhs);
}

extern "C" int tm_loop_contract(const tm_lattice* L, const void* a_full, const void* b_full, int prec, int nrhs, double* out,
                                void* workspace, void* stream)
{
    if (!L || !a_full || !b_full || !out || !workspace || !valid_prec(prec) || nrhs < 1) return TM_ERR_ARG;
    if (!aligned256(a_full) || !aligned256(b_full) || !aligned256(out) || !aligned256(workspace)) return TM_ERR_LAYOUT;
    return loop_contract(L->g, a_full, b_full, prec, nrhs, out, workspace, (cudaStream_t)stream);
}

extern "C" int tm_loop_contract_ex(const tm_lattice* L, const void* a_full, const void* b_full, int prec, int nrhs, int g5_left,
                                   int g5_right, double scale_re, double scale_im, double* out, void* workspace, void* stream)
{
    if (!L || !a_full || !b_full || !out || !workspace || !valid_prec(prec) || nrhs < 1) return TM_ERR_ARG;
    if (!aligned256(a_full) || !aligned256(b_full) || !aligned256(out) || !aligned256(workspace)) return TM_ERR_LAYOUT;
    return loop_contract_ex(L->g, a_full, b_full, prec, nrhs, out, workspace, g5_left != 0, g5_right != 0, scale_re, scale_im,
                            (cudaStream_t)stream);
}

/* ---- the loop contraction for callers that cannot allocate (tm.h: tm_loop_contract_static) --------------------------------
 * Same two kernels as tm_loop_contract; the per-block partial sums go to a file-scope device array instead of a caller workspace.
 * In host code `g_loop_scratch` is only the host-side stand-in of the symbol, NOT a device address: the address is looked up once
 * per device (with that device current) by cudaGetSymbolAddress and that pointer is what the kernels get. */
static __device__ __align__(256) unsigned char g_loop_scratch[TM_LOOP_STATIC_BYTES];

static int loop_scratch_ptr(void** out)
{
    constexpr int MAX_DEV = 64;
    static std::mutex mu;
    static void* ptrs[MAX_DEV] = {};
    int dev = -1;
    TM_CUDA_CHECK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEV) return TM_ERR_ARG;
    std::lock_guard<std::mutex> lk(mu);
    if (ptrs[dev] == nullptr) {
        void* p = nullptr;
        TM_CUDA_CHECK(cudaGetSymbolAddress(&p, g_loop_scratch));
        if (p == nullptr) return TM_ERR_CUDA;
        ptrs[dev] = p;
    }
    *out = ptrs[dev];
    return TM_OK;
}

extern "C" int tm_loop_contract_static(const tm_lattice* L, const void* a_full, const void* b_full, int prec, int nrhs, double* out,
                                       void* stream)
{
    if (!L || !a_full || !b_full || !out || !valid_prec(prec) || nrhs < 1) return TM_ERR_ARG;
    if (!aligned256(a_full) || !aligned256(b_full) || !aligned256(out)) return TM_ERR_LAYOUT;
    if (loop_workspace_bytes(L->g, nrhs) > (size_t)TM_LOOP_STATIC_BYTES) return TM_ERR_STATIC_LIMIT;
    void* scratch = nullptr;
    const int rc = loop_scratch_ptr(&scratch);
    if (rc != TM_OK) return rc;
    // nothing has to start at zero: loop_partial_kernel writes every partial that loop_final_kernel reads
    return loop_contract(L->g, a_full, b_full, prec, nrhs, out, scratch, (cudaStream_t)stream);
}

/* single-time-slice contraction, used with time-diluted sources */
extern "C" int tm_loop_contract_slice(const tm_lattice* L, const void* a_full, const void* b_full, int prec, int nrhs, int t0,
                                      double* out, void* workspace, void* stream)
{
    if (!L || !a_full || !b_full || !out || !workspace || !valid_prec(prec) || nrhs < 1) return TM_ERR_ARG;
    if (t0 < 0 || t0 >= L->g.T) return TM_ERR_ARG;
    if (!aligned256(a_full) || !aligned256(b_full) || !aligned256(out) || !aligned256(workspace)) return TM_ERR_LAYOUT;
    return loop_contract_range(L->g, a_full, b_full, prec, nrhs, out, workspace, 0, 0, 1.0, 0.0, t0, 1, (cudaStream_t)stream);
}
