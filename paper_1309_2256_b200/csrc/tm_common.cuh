// tm_common.cuh -- host/device plumbing shared by the library's translation units (CUDA path only;
// nothing here is used by, or uses, the oracle).
#pragma once
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/tm.h"

namespace tmk {

// n / d for 0 <= n < 2^31 by multiply-high (Granlund-Montgomery round-up method)
struct FastDiv {
    uint32_t d, m, s;
    __host__ void init(uint32_t d_)
    {
        d = d_;
        s = 0;
        while ((1u << s) < d) ++s;
        m = (uint32_t)(((uint64_t(1) << 32) * ((uint64_t(1) << s) - d)) / d + 1);
    }
    __device__ __forceinline__ uint32_t div(uint32_t n) const { return (__umulhi(m, n) + n) >> s; }
    __device__ __forceinline__ void divmod(uint32_t n, uint32_t& q, uint32_t& r) const
    {
        q = div(n);
        r = n - q * d;
    }
};

// geometry as the kernels see it
struct Geo {
    int X, Y, Z, T;
    int Xh;      // X/2
    int Vh;      // sites per parity
    int V3h;     // X*Y*Z/2 = checkerboard sites per time slice
    int XhY;     // Xh*Y
    int ap;      // antiperiodic in time
    FastDiv dXh, dY, dZ;
};

} // namespace tmk

struct tm_lattice {
    tmk::Geo g;
    long long V;
};

namespace tmk {

// ---- error / launch bookkeeping (tm_api.cu) ----
void note_launch(unsigned long long n = 1);
int cuda_fail(cudaError_t e, const char* where);
#define TM_CUDA_CHECK(expr)                                        \
    do {                                                           \
        cudaError_t e__ = (expr);                                  \
        if (e__ != cudaSuccess) return tmk::cuda_fail(e__, #expr);  \
    } while (0)
#define TM_LAUNCH_CHECK(what)                                      \
    do {                                                           \
        tmk::note_launch();                                         \
        cudaError_t e__ = cudaGetLastError();                      \
        if (e__ != cudaSuccess) return tmk::cuda_fail(e__, what);   \
    } while (0)

static inline bool aligned256(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 255u) == 0; }
static inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; } // one-parity views
static inline size_t round256(size_t n) { return (n + 255) & ~size_t(255); }

// bytes of one single-parity spinor / one (parity,mu) link block
static inline size_t spinor_parity_bytes(const Geo& g, int prec) { return (size_t)g.Vh * 24 * prec + (prec == 2 ? (size_t)g.Vh * 4 : 0); }
static inline size_t link_block_bytes(const Geo& g, int prec, int recon) { return (size_t)g.Vh * (recon % 100) * prec; }

static inline bool valid_prec(int p) { return p == 8 || p == 4 || p == 2; }
static inline bool valid_recon(int r) { return r == 18 || r == 12 || r == 8 || r == 118 || r == 112 || r == 218 || r == 212; }
// TM_RECON_*_FIX16 (reals + 100) means 16-bit fixed-point link words and exists for 16-bit storage only: plain recon otherwise.
// TM_RECON_*_TG (reals + 200) declares temporal gauge; the field is stored like the plain one, fp64 kernels ignore the declaration.
static inline int link_recon(int prec, int recon) { return recon >= 200 ? (prec == 8 ? recon - 200 : recon) : (prec == 2 ? recon : recon % 100); }
static inline int stored_recon(int prec, int recon) { recon = link_recon(prec, recon); return recon >= 200 ? recon - 200 : recon; }

// ---- internal launchers (defined in their own .cu files) ----
struct DslashParams {
    const void* gauge; // packed links
    void* out;
    const void* in;
    const void* x;     // may be null
    int out_parity;
    int dagger;
    double pq[4];      // out = (p0 + i p1 g5) x + (q0 + i q1 g5) D in
    int nrhs;
    size_t rhs_stride_out, rhs_stride_in, rhs_stride_x; // bytes between consecutive right-hand sides
    const unsigned char* active; // optional per-rhs device flags: rhs with active[r] == 0 is skipped (may be null)
    const void* link_cache = nullptr; // optional: link_cache_build() output for this gauge field (fp32 / fp16, nrhs > 6)
    // optional fused reduction: dot_partial[rhs][ceil(Vh/32)] = per-warp sums of Re <dot_with, out> (|out|^2 if dot_with is null)
    const void* dot_with = nullptr;
    size_t dot_stride = 0;
    double* dot_partial = nullptr;
    // optional fused axpy: out = axpy_y - coef[rhs] * (epilogue result), coef = device doubles at axpy_coef + rhs * axpy_coef_stride
    const void* axpy_y = nullptr;
    size_t axpy_y_stride = 0;
    const void* axpy_coef = nullptr;
    size_t axpy_coef_stride = 0;
};
int launch_dslash(const Geo& g, int prec, int recon, const DslashParams& p, cudaStream_t st);
void kind_pq(int kind, int dagger, double kappa, double mu, double pq[4]);
// fp32 tile images of all links (both parities) for the multi-rhs kernel; 0 bytes for fp64
size_t link_cache_bytes(const Geo& g, int prec);
int link_cache_build(const Geo& g, int prec, int recon, const void* gauge, void* cache, cudaStream_t st);
int mdagm_apply(const Geo& g, const void* gauge, int prec, int recon, void* out, size_t out_stride, const void* in,
                size_t in_stride, void* tmp, int parity, double kappa, double mu, int nrhs, const unsigned char* active,
                cudaStream_t st, const void* link_cache = nullptr, double* dot_partial = nullptr);
int spinor_pack_any(const Geo& g, long long V, int prec, int mode, const double* src, double* dst, const unsigned char* codes,
                    void* packed, int nrhs, cudaStream_t st);
int loop_contract(const Geo& g, const void* a_full, const void* b_full, int prec, int nrhs, double* out, void* workspace,
                  cudaStream_t st);
int loop_contract_ex(const Geo& g, const void* a_full, const void* b_full, int prec, int nrhs, double* out, void* workspace,
                     int g5_left, int g5_right, double scale_re, double scale_im, cudaStream_t st);
size_t loop_workspace_bytes(const Geo& g, int nrhs);
int loop_contract_range(const Geo& g, const void* a_full, const void* b_full, int prec, int nrhs, double* out, void* workspace,
                        int g5_left, int g5_right, double scale_re, double scale_im, int t0, int nt, cudaStream_t st);
void kernel_timing_begin(cudaStream_t st);
void kernel_timing_end(cudaStream_t st);

} // namespace tmk
