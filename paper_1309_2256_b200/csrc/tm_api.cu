// tm_api.cu -- C ABI entry points: geometry, sizes, errors, instrumentation, tm_dslash, tm_MdagM.
#include "tm_common.cuh"
#include <atomic>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

namespace tmk {

static std::atomic<unsigned long long> g_launches{0};
static thread_local char g_cuda_err[512] = "";

void note_launch(unsigned long long n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

int cuda_fail(cudaError_t e, const char* where)
{
    snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s (%s)", where, cudaGetErrorName(e), cudaGetErrorString(e));
    return TM_ERR_CUDA;
}

// ---- optional per-launch event timing of the dslash family ----
static bool g_timing = false;
static std::mutex g_timing_mu;
static std::vector<cudaEvent_t> g_ev_pool; // pairs: begin, end
static size_t g_ev_used = 0;

void kernel_timing_begin(cudaStream_t st)
{
    if (!g_timing) return;
    std::lock_guard<std::mutex> lk(g_timing_mu);
    if (g_ev_used + 2 > g_ev_pool.size()) {
        cudaEvent_t a, b;
        cudaEventCreate(&a);
        cudaEventCreate(&b);
        g_ev_pool.push_back(a);
        g_ev_pool.push_back(b);
    }
    cudaEventRecord(g_ev_pool[g_ev_used], st);
}

void kernel_timing_end(cudaStream_t st)
{
    if (!g_timing) return;
    std::lock_guard<std::mutex> lk(g_timing_mu);
    cudaEventRecord(g_ev_pool[g_ev_used + 1], st);
    g_ev_used += 2;
}

template <int PREC, int RECON>
int launch_dslash_t(const Geo& g, const DslashParams& p, cudaStream_t st);
#define TM_DECL(P, R) template <> int launch_dslash_t<P, R>(const Geo&, const DslashParams&, cudaStream_t);
TM_DECL(8, 18) TM_DECL(8, 12) TM_DECL(8, 8) TM_DECL(4, 18) TM_DECL(4, 12) TM_DECL(4, 8) TM_DECL(2, 18) TM_DECL(2, 12) TM_DECL(2, 8)
TM_DECL(2, 118) TM_DECL(2, 112) TM_DECL(4, 218) TM_DECL(4, 212) TM_DECL(2, 218) TM_DECL(2, 212)
#undef TM_DECL

template <int PREC, int RECON>
int link_cache_build_t(const Geo& g, const void* gauge, void* cache, cudaStream_t st);
#define TM_DECL_LC(P, R) template <> int link_cache_build_t<P, R>(const Geo&, const void*, void*, cudaStream_t);
TM_DECL_LC(4, 18) TM_DECL_LC(4, 12) TM_DECL_LC(4, 8) TM_DECL_LC(2, 18) TM_DECL_LC(2, 12) TM_DECL_LC(2, 8) TM_DECL_LC(2, 118) TM_DECL_LC(2, 112)

// sizeof(TileSmem<32>) = 8*32*4 + 8*4*32*16 + 8*32*8 bytes per 32-site tile, both parities
size_t link_cache_bytes(const Geo& g, int prec)
{
    if (prec == 8) return 0;
    return round256((size_t)2 * ((g.Vh + 31) / 32) * 19456);
}

int link_cache_build(const Geo& g, int prec, int recon, const void* gauge, void* cache, cudaStream_t st)
{
    recon = stored_recon(prec, recon);
    if (prec == 4) return recon == 18 ? link_cache_build_t<4, 18>(g, gauge, cache, st) : recon == 12 ? link_cache_build_t<4, 12>(g, gauge, cache, st) : link_cache_build_t<4, 8>(g, gauge, cache, st);
    if (prec == 2 && recon >= 100) return recon == 118 ? link_cache_build_t<2, 118>(g, gauge, cache, st) : link_cache_build_t<2, 112>(g, gauge, cache, st);
    if (prec == 2) return recon == 18 ? link_cache_build_t<2, 18>(g, gauge, cache, st) : recon == 12 ? link_cache_build_t<2, 12>(g, gauge, cache, st) : link_cache_build_t<2, 8>(g, gauge, cache, st);
    return TM_ERR_ARG;
}

int launch_dslash(const Geo& g, int prec, int recon, const DslashParams& p, cudaStream_t st)
{
    recon = link_recon(prec, recon); // the fixed-point flag exists for 16-bit links only (tm.h)
    if (recon >= 200) { // temporal gauge declared: the single-rhs fp32 / fp16 kernels skip the unit links, the others read them
        if (p.nrhs == 1) {
            if (prec == 4) return recon == 218 ? launch_dslash_t<4, 218>(g, p, st) : launch_dslash_t<4, 212>(g, p, st);
            return recon == 218 ? launch_dslash_t<2, 218>(g, p, st) : launch_dslash_t<2, 212>(g, p, st);
        }
        recon -= 200;
    }
    if (prec == 8) return recon == 18 ? launch_dslash_t<8, 18>(g, p, st) : recon == 12 ? launch_dslash_t<8, 12>(g, p, st) : launch_dslash_t<8, 8>(g, p, st);
    if (prec == 4) return recon == 18 ? launch_dslash_t<4, 18>(g, p, st) : recon == 12 ? launch_dslash_t<4, 12>(g, p, st) : launch_dslash_t<4, 8>(g, p, st);
    if (recon >= 100) return recon == 118 ? launch_dslash_t<2, 118>(g, p, st) : launch_dslash_t<2, 112>(g, p, st);
    return recon == 18 ? launch_dslash_t<2, 18>(g, p, st) : recon == 12 ? launch_dslash_t<2, 12>(g, p, st) : launch_dslash_t<2, 8>(g, p, st);
}

} // namespace tmk

using namespace tmk;

extern "C" int tm_version(void) { return TM_VERSION; }

extern "C" const char* tm_strerror(int s)
{
    switch (s) {
    case TM_OK: return "ok";
    case TM_ERR_ARG: return "invalid argument";
    case TM_ERR_LAYOUT: return "bad lattice dimensions, alignment or workspace size";
    case TM_ERR_NOT_SU3: return "gauge link is not SU(3) within su3_tol (required for 12- and 8-real storage)";
    case TM_ERR_NOT_TGAUGE: return "a temporal link of a slice t < T-1 is not the unit matrix (field declared in temporal gauge)";
    case TM_ERR_RECON8: return "a gauge link lies where the 8-real parametrisation is singular (|U01|^2 + |U02|^2 < 1e-6)";
    case TM_ERR_CUDA: return "CUDA runtime error (see tm_last_cuda_error)";
    case TM_ERR_BREAKDOWN: return "CG breakdown (<p,Ap> <= 0 or NaN)";
    case TM_ERR_MAXITER: return "CG reached max_iter before the requested tolerance";
    case TM_ERR_STATIC_LIMIT: return "tm_loop_contract_static: nrhs * T * blocks needs more than the TM_LOOP_STATIC_BYTES (8 MiB) static scratch array; use tm_loop_contract with a workspace";
    default: return "unknown status";
    }
}

extern "C" const char* tm_last_cuda_error(void) { return g_cuda_err; }
extern "C" unsigned long long tm_launch_count(void) { return g_launches.load(); }

namespace tmk { const char* lc_kernel_signature(); }
extern "C" const char* tm_kernel_signature(void) { return tmk::lc_kernel_signature(); }

extern "C" int tm_kernel_timing_enable(int on)
{
    std::lock_guard<std::mutex> lk(g_timing_mu);
    g_timing = on != 0;
    return TM_OK;
}

extern "C" int tm_kernel_timing_read(double* ms_total, long long* launches, int reset)
{
    TM_CUDA_CHECK(cudaDeviceSynchronize());
    std::lock_guard<std::mutex> lk(g_timing_mu);
    double tot = 0;
    for (size_t k = 0; k + 1 < g_ev_used; k += 2) {
        float ms = 0;
        TM_CUDA_CHECK(cudaEventElapsedTime(&ms, g_ev_pool[k], g_ev_pool[k + 1]));
        tot += ms;
    }
    if (ms_total) *ms_total = tot;
    if (launches) *launches = (long long)(g_ev_used / 2);
    if (reset) g_ev_used = 0;
    return TM_OK;
}

extern "C" int tm_lattice_create(tm_lattice** out, const int dims[4], int antiperiodic_t)
{
    if (!out || !dims) return TM_ERR_ARG;
    for (int k = 0; k < 4; ++k)
        if (dims[k] < 4 || (dims[k] & 1)) return TM_ERR_LAYOUT;
    const long long V = (long long)dims[0] * dims[1] * dims[2] * dims[3];
    if (V / 2 > (1ll << 27)) return TM_ERR_LAYOUT; // 32-bit element indexing inside the kernels
    tm_lattice* L = new (std::nothrow) tm_lattice;
    if (!L) return TM_ERR_ARG;
    Geo& g = L->g;
    g.X = dims[0]; g.Y = dims[1]; g.Z = dims[2]; g.T = dims[3];
    g.Xh = g.X / 2;
    g.Vh = (int)(V / 2);
    g.V3h = g.Xh * g.Y * g.Z;
    g.XhY = g.Xh * g.Y;
    g.ap = antiperiodic_t ? 1 : 0;
    g.dXh.init(g.Xh); g.dY.init(g.Y); g.dZ.init(g.Z);
    L->V = V;
    *out = L;
    return TM_OK;
}

extern "C" void tm_lattice_destroy(tm_lattice* L) { delete L; }

extern "C" size_t tm_gauge_bytes(const tm_lattice* L, int prec, int recon)
{
    if (!L || !valid_prec(prec) || !valid_recon(recon)) return 0;
    return 8 * link_block_bytes(L->g, prec, recon);
}

extern "C" size_t tm_spinor_bytes(const tm_lattice* L, int prec, int full, int nrhs)
{
    if (!L || !valid_prec(prec) || nrhs < 1) return 0;
    return spinor_parity_bytes(L->g, prec) * (full ? 2 : 1) * (size_t)nrhs;
}

static int dslash_common(const tm_lattice* L, const void* gauge, int prec, int recon, void* out, const void* in, const void* x,
                         int out_parity, int dagger, const double pq[4], int nrhs, void* stream)
{
    if (!L || !gauge || !out || !in || !valid_prec(prec) || !valid_recon(recon)) return TM_ERR_ARG;
    if (out == in || nrhs < 1 || nrhs > TM_MAX_NRHS || (out_parity & ~1)) return TM_ERR_ARG;
    if (!x && (pq[0] != 0.0 || pq[1] != 0.0)) return TM_ERR_ARG;
    // one-parity spinors may be views into a full-lattice buffer (odd block at + parity bytes): 16-byte chunks must stay aligned
    if (!aligned256(gauge) || !aligned16(out) || !aligned16(in) || (x && !aligned16(x))) return TM_ERR_LAYOUT;
    DslashParams p;
    p.gauge = gauge; p.out = out; p.in = in;
    p.x = (pq[0] != 0.0 || pq[1] != 0.0) ? x : nullptr;
    p.out_parity = out_parity; p.dagger = dagger ? 1 : 0;
    for (int k = 0; k < 4; ++k) p.pq[k] = pq[k];
    p.nrhs = nrhs;
    p.rhs_stride_out = p.rhs_stride_in = p.rhs_stride_x = spinor_parity_bytes(L->g, prec);
    p.active = nullptr;
    return launch_dslash(L->g, prec, recon, p, (cudaStream_t)stream);
}

namespace tmk {
void kind_pq(int kind, int dagger, double kappa, double mu, double pq[4])
{
    const double a = 2.0 * kappa * mu * (dagger ? -1.0 : 1.0);
    pq[0] = pq[1] = pq[2] = pq[3] = 0.0;
    if (kind == TM_KIND_PLAIN) { pq[2] = 1.0; }
    else if (kind == TM_KIND_TWIST_INV) { pq[2] = 1.0 / (1.0 + a * a); pq[3] = -a / (1.0 + a * a); } // R^-1 = (1 - i a g5)/(1+a^2)
    else { pq[0] = 1.0; pq[1] = a; pq[2] = -kappa * kappa; }                                          // R x - kappa^2 D in
}
} // namespace tmk

extern "C" int tm_dslash_general(const tm_lattice* L, const void* gauge, int prec, int recon, void* out, const void* in,
                                 const void* x, int out_parity, int dagger, const double pq[4], int nrhs, void* stream)
{
    if (!pq) return TM_ERR_ARG;
    return dslash_common(L, gauge, prec, recon, out, in, x, out_parity, dagger, pq, nrhs, stream);
}

extern "C" int tm_dslash(const tm_lattice* L, const void* gauge, int prec, int recon, void* out, const void* in, const void* x,
                         int out_parity, int dagger, int kind, double kappa, double mu, int nrhs, void* stream)
{
    if (kind < 0 || kind > 2) return TM_ERR_ARG;
    if (kind == TM_KIND_XPAY_TWIST && !x) return TM_ERR_ARG;
    double pq[4];
    kind_pq(kind, dagger, kappa, mu, pq);
    return dslash_common(L, gauge, prec, recon, out, in, x, out_parity, dagger, pq, nrhs, stream);
}

namespace tmk {
// M_pc^dag M_pc on `parity` with explicit strides/active flags (shared by tm_MdagM and the CG driver)
int mdagm_apply(const Geo& g, const void* gauge, int prec, int recon, void* out, size_t out_stride, const void* in,
                size_t in_stride, void* tmp, int parity, double kappa, double mu, int nrhs, const unsigned char* active,
                cudaStream_t st, const void* link_cache, double* dot_partial)
{
    const size_t pb = spinor_parity_bytes(g, prec);
    char* t1 = static_cast<char*>(tmp);
    char* t2 = t1 + pb * nrhs;
    DslashParams p;
    p.gauge = gauge; p.nrhs = nrhs; p.active = active; p.link_cache = link_cache;
    p.rhs_stride_out = p.rhs_stride_in = p.rhs_stride_x = pb;
    int rc;
    // t1 = R^-1 D_{pbar p} in
    p.out = t1; p.in = in; p.x = nullptr; p.out_parity = 1 - parity; p.dagger = 0;
    p.rhs_stride_in = in_stride;
    kind_pq(TM_KIND_TWIST_INV, 0, kappa, mu, p.pq);
    if ((rc = launch_dslash(g, prec, recon, p, st)) != TM_OK) return rc;
    // t2 = R in - kappa^2 D_{p pbar} t1 = M_pc in
    p.out = t2; p.in = t1; p.x = in; p.out_parity = parity;
    p.rhs_stride_in = pb; p.rhs_stride_x = in_stride;
    kind_pq(TM_KIND_XPAY_TWIST, 0, kappa, mu, p.pq);
    // <in, M_pc^dag M_pc in> = |M_pc in|^2: the CG's <p,Ap> falls out of this launch's epilogue with no extra load
    p.dot_partial = dot_partial;
    if ((rc = launch_dslash(g, prec, recon, p, st)) != TM_OK) return rc;
    p.dot_partial = nullptr;
    // t1 = R(-a)^-1 D^dag_{pbar p} t2
    p.out = t1; p.in = t2; p.x = nullptr; p.out_parity = 1 - parity; p.dagger = 1;
    p.rhs_stride_x = pb;
    kind_pq(TM_KIND_TWIST_INV, 1, kappa, mu, p.pq);
    if ((rc = launch_dslash(g, prec, recon, p, st)) != TM_OK) return rc;
    // out = R(-a) t2 - kappa^2 D^dag_{p pbar} t1 = M_pc^dag t2
    p.out = out; p.in = t1; p.x = t2; p.out_parity = parity;
    p.rhs_stride_out = out_stride;
    kind_pq(TM_KIND_XPAY_TWIST, 1, kappa, mu, p.pq);
    return launch_dslash(g, prec, recon, p, st);
}
} // namespace tmk

extern "C" int tm_MdagM(const tm_lattice* L, const void* gauge, int prec, int recon, void* out, const void* in, void* tmp,
                        int parity, double kappa, double mu, int nrhs, void* stream)
{
    if (!L || !gauge || !out || !in || !tmp || !valid_prec(prec) || !valid_recon(recon)) return TM_ERR_ARG;
    if (nrhs < 1 || nrhs > TM_MAX_NRHS || (parity & ~1)) return TM_ERR_ARG;
    if (!aligned256(gauge) || !aligned16(out) || !aligned16(in) || !aligned256(tmp)) return TM_ERR_LAYOUT;
    const size_t pb = spinor_parity_bytes(L->g, prec);
    return mdagm_apply(L->g, gauge, prec, recon, out, pb, in, pb, tmp, parity, kappa, mu, nrhs, nullptr, (cudaStream_t)stream);
}
