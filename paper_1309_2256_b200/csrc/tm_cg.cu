// tm_cg.cu -- a6 / a7 of SURVEY.md 8(a): CG on the even-even Schur system, truncated LP mode batched over
// right-hand sides, mixed-precision HP mode with reliable updates, and the host-buffer TSM batch entry point.
//
//   b' = eta_e + kappa Dslash_eo R^-1 eta_o;  b'' = M_pc^dag b';  CG on A = M_pc^dag M_pc, x0 = 0;
//   s_e = x;  s_o = R^-1 (eta_o + kappa Dslash_oe s_e)                 (PAPER.md:373-381 Eq. A2, A4 as corrected
//   in DESIGN.md reading 6; PAPER.md:67 for the truncation rule)
#include "tm_blas.cuh"
#include <cmath>
#include <cstring>
#include <new>
#include <vector>

namespace tmk {

template <typename F>
static inline int by_prec(int prec, F&& f)
{
    if (prec == 8) return f(std::integral_constant<int, 8>());
    if (prec == 4) return f(std::integral_constant<int, 4>());
    return f(std::integral_constant<int, 2>());
}

static inline VecArg V_(void* p, size_t stride) { return VecArg{static_cast<char*>(p), stride}; }
static inline VecArg V_(const void* p, size_t stride) { return VecArg{static_cast<char*>(const_cast<void*>(p)), stride}; }

static int k_twist(const Geo& g, int prec, VecArg out, VecArg in, double c0, double c1, int nrhs, cudaStream_t st)
{
    dim3 grid(blas_blocks(g.Vh), nrhs);
    return by_prec(prec, [&](auto P) {
        twist_kernel<decltype(P)::value><<<grid, BLAS_THREADS, 0, st>>>(g.Vh, out, in, c0, c1);
        TM_LAUNCH_CHECK("twist_kernel");
        return (int)TM_OK;
    });
}

template <int FIN>
static int k_norm2(const Geo& g, int prec, VecArg v, const BlasCtx& c, int nrhs, cudaStream_t st)
{
    dim3 grid(blas_blocks(g.Vh), nrhs);
    return by_prec(prec, [&](auto P) {
        norm2_kernel<decltype(P)::value, FIN><<<grid, BLAS_THREADS, 0, st>>>(g.Vh, v, c);
        TM_LAUNCH_CHECK("norm2_kernel");
        return (int)TM_OK;
    });
}

// out(po) = in(pi) [and out2]
static int k_convert(const Geo& g, int po, int pi, VecArg out, VecArg out2, VecArg in, int nrhs, cudaStream_t st)
{
    dim3 grid(blas_blocks(g.Vh), nrhs);
    return by_prec(po, [&](auto PO) {
        return by_prec(pi, [&](auto PI) {
            convert_kernel<decltype(PO)::value, decltype(PI)::value><<<grid, BLAS_THREADS, 0, st>>>(g.Vh, out, out2, in);
            TM_LAUNCH_CHECK("convert_kernel");
            return (int)TM_OK;
        });
    });
}

template <int REDUCE>
static int k_axpby(const Geo& g, int py, int px, VecArg y, VecArg x, double a, double b, const BlasCtx& c, int nrhs, cudaStream_t st)
{
    dim3 grid(blas_blocks(g.Vh), nrhs);
    return by_prec(py, [&](auto PY) {
        return by_prec(px, [&](auto PX) {
            axpby_kernel<decltype(PY)::value, decltype(PX)::value, REDUCE><<<grid, BLAS_THREADS, 0, st>>>(g.Vh, y, x, a, b, c);
            TM_LAUNCH_CHECK("axpby_kernel");
            return (int)TM_OK;
        });
    });
}

static int k_cg_iter(const Geo& g, const void* gauge, int prec, int recon, VecArg x, VecArg r, VecArg p, VecArg Ap, void* tmp,
                     double kappa, double mu, const BlasCtx& c, int nrhs, bool do_update_p, cudaStream_t st,
                     const void* link_cache = nullptr)
{
    int rc = mdagm_apply(g, gauge, prec, recon, Ap.p, Ap.stride, p.p, p.stride, tmp, 0, kappa, mu, nrhs, c.active, st, link_cache);
    if (rc != TM_OK) return rc;
    dim3 grid(blas_blocks(g.Vh), nrhs);
    return by_prec(prec, [&](auto P) {
        constexpr int PR = decltype(P)::value;
        dot_pAp_kernel<PR><<<grid, BLAS_THREADS, 0, st>>>(g.Vh, p, Ap, c);
        TM_LAUNCH_CHECK("dot_pAp_kernel");
        update_xr_kernel<PR><<<grid, BLAS_THREADS, 0, st>>>(g.Vh, x, r, p, Ap, c);
        TM_LAUNCH_CHECK("update_xr_kernel");
        if (do_update_p) {
            update_p_kernel<PR><<<grid, BLAS_THREADS, 0, st>>>(g.Vh, p, r, c);
            TM_LAUNCH_CHECK("update_p_kernel");
        }
        return (int)TM_OK;
    });
}

// One truncated-CG iteration (LP mode) with the reductions and the residual update fused into the operator:
//   t1 = R^-1 D p;  t2 = M_pc p, partials of |t2|^2 = <p, A p>;  [finalize -> alpha]
//   t1 = R(-a)^-1 D^dag t2;  r = r - alpha (R(-a) t2 - kappa^2 D^dag t1), partials of |r|^2;  [finalize -> beta, convergence]
//   x += alpha p, p = r + beta p.
// A p is never written to memory; the only vector kernel left moves 5 one-parity spinors per rhs (11 before).
// pin / rin: where this iteration READS its search direction and residual (the stacks p / r themselves from iteration 1 on; the
// right-hand side b in iteration 0, where p_0 = r_0 = b: the solver makes no copies of b).
static int k_cg_iter_fused(const Geo& g, const void* gauge, int prec, int recon, VecArg x, VecArg r, VecArg p, VecArg rin, VecArg pin,
                           void* tmp, double kappa, double mu, const BlasCtx& c, double* partial, int nrhs, int iter, cudaStream_t st,
                           const void* link_cache, bool do_xp = true)
{
    const size_t pb = spinor_parity_bytes(g, prec);
    char* t1 = static_cast<char*>(tmp);
    char* t2 = t1 + pb * nrhs;
    const int ngroups = (g.Vh + 31) / 32;
    DslashParams d;
    d.gauge = gauge; d.nrhs = nrhs; d.active = c.active; d.link_cache = link_cache;
    d.rhs_stride_out = d.rhs_stride_in = d.rhs_stride_x = pb;
    int rc;
    d.out = t1; d.in = pin.p; d.x = nullptr; d.out_parity = 1; d.dagger = 0; d.rhs_stride_in = pin.stride;
    kind_pq(TM_KIND_TWIST_INV, 0, kappa, mu, d.pq);
    if ((rc = launch_dslash(g, prec, recon, d, st)) != TM_OK) return rc;
    d.out = t2; d.in = t1; d.x = pin.p; d.out_parity = 0; d.rhs_stride_in = pb; d.rhs_stride_x = pin.stride;
    kind_pq(TM_KIND_XPAY_TWIST, 0, kappa, mu, d.pq);
    d.dot_partial = partial;
    if ((rc = launch_dslash(g, prec, recon, d, st)) != TM_OK) return rc;
    d.dot_partial = nullptr;
    dot_finalize_kernel<FIN_PAP><<<nrhs, FIN_THREADS, 0, st>>>(partial, ngroups, c);
    TM_LAUNCH_CHECK("dot_finalize_kernel");
    d.out = t1; d.in = t2; d.x = nullptr; d.out_parity = 1; d.dagger = 1; d.rhs_stride_x = pb;
    kind_pq(TM_KIND_TWIST_INV, 1, kappa, mu, d.pq);
    if ((rc = launch_dslash(g, prec, recon, d, st)) != TM_OK) return rc;
    d.out = r.p; d.in = t1; d.x = t2; d.out_parity = 0; d.rhs_stride_out = r.stride;
    kind_pq(TM_KIND_XPAY_TWIST, 1, kappa, mu, d.pq);
    d.axpy_y = rin.p; d.axpy_y_stride = rin.stride;
    d.axpy_coef = &c.scal[0].alpha; d.axpy_coef_stride = sizeof(CgScal);
    d.dot_partial = partial;
    if ((rc = launch_dslash(g, prec, recon, d, st)) != TM_OK) return rc;
    dot_finalize_kernel<FIN_RR><<<nrhs, FIN_THREADS, 0, st>>>(partial, ngroups, c);
    TM_LAUNCH_CHECK("dot_finalize_kernel");
    if (!do_xp) return TM_OK; // the caller keeps the search directions in a ring and forms x afterwards
    dim3 grid(blas_blocks(g.Vh), nrhs);
    return by_prec(prec, [&](auto P) {
        update_xp_kernel<decltype(P)::value><<<grid, BLAS_THREADS, 0, st>>>(g.Vh, x, p, pin, r, c, iter);
        TM_LAUNCH_CHECK("update_xp_kernel");
        return (int)TM_OK;
    });
}

static int k_update_p(const Geo& g, int prec, VecArg p, VecArg r, const BlasCtx& c, int nrhs, cudaStream_t st)
{
    dim3 grid(blas_blocks(g.Vh), nrhs);
    return by_prec(prec, [&](auto P) {
        update_p_kernel<decltype(P)::value><<<grid, BLAS_THREADS, 0, st>>>(g.Vh, p, r, c);
        TM_LAUNCH_CHECK("update_p_kernel");
        return (int)TM_OK;
    });
}

// pinned host ring for the pipelined convergence poll of cg_lp_truncated: library-owned host memory, one ring per (host thread,
// device), created on first use and released when the thread ends; a failed creation leaves nothing behind.
struct PollRing {
    static constexpr int DEPTH = 4;
    unsigned char* flags = nullptr; // [DEPTH][TM_MAX_NRHS], pinned
    cudaEvent_t ev[DEPTH] = {};
    int nev = 0;
    int device = -1;
    bool create(int dev)
    {
        device = dev;
        if (cudaHostAlloc(reinterpret_cast<void**>(&flags), DEPTH * TM_MAX_NRHS, cudaHostAllocDefault) != cudaSuccess) {
            flags = nullptr;
            return false;
        }
        for (nev = 0; nev < DEPTH; ++nev)
            if (cudaEventCreateWithFlags(&ev[nev], cudaEventDisableTiming) != cudaSuccess) {
                destroy();
                return false;
            }
        return true;
    }
    void destroy()
    {
        for (int i = 0; i < nev; ++i) cudaEventDestroy(ev[i]);
        nev = 0;
        if (flags) cudaFreeHost(flags);
        flags = nullptr;
    }
};
struct PollRings {
    std::vector<PollRing*> rings; // one per device this thread has solved on
    ~PollRings()
    {
        for (PollRing* r : rings) {
            // at thread exit the context may already be gone; the calls then fail harmlessly
            int cur = -1;
            if (cudaGetDevice(&cur) == cudaSuccess && cudaSetDevice(r->device) == cudaSuccess) {
                r->destroy();
                cudaSetDevice(cur);
            }
            delete r;
        }
    }
};
static PollRing* poll_ring()
{
    static thread_local PollRings mine;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return nullptr;
    for (PollRing* r : mine.rings)
        if (r->device == dev) return r;
    PollRing* r = new (std::nothrow) PollRing;
    if (!r) return nullptr;
    if (!r->create(dev)) { // nothing half-built survives: the next call starts from scratch
        delete r;
        return nullptr;
    }
    mine.rings.push_back(r);
    return r;
}

// carve a workspace
struct Carver {
    char* base;
    size_t off = 0, cap;
    Carver(void* p, size_t c) : base(static_cast<char*>(p)), cap(c) {}
    void* take(size_t n)
    {
        void* r = base + off;
        off += round256(n);
        return r;
    }
    bool ok() const { return off <= cap; }
};

static size_t ctx_bytes(int nrhs)
{
    return round256(sizeof(CgScal) * nrhs) + round256(nrhs) + round256(sizeof(unsigned int) * nrhs) +
           round256(sizeof(double) * BLAS_MAX_BLOCKS * nrhs);
}

static BlasCtx carve_ctx(Carver& cv, int nrhs)
{
    BlasCtx c;
    c.scal = static_cast<CgScal*>(cv.take(sizeof(CgScal) * nrhs));
    c.active = static_cast<unsigned char*>(cv.take(nrhs));
    c.tickets = static_cast<unsigned int*>(cv.take(sizeof(unsigned int) * nrhs));
    c.partials = static_cast<double*>(cv.take(sizeof(double) * BLAS_MAX_BLOCKS * nrhs));
    return c;
}

static int init_ctx(const BlasCtx& c, const tm_cg_params* p, int nrhs, cudaStream_t st)
{
    std::vector<CgScal> h(nrhs);
    for (auto& s : h) {
        memset(&s, 0, sizeof(s));
        s.tol2 = p->tol * p->tol;
        s.max_iter = p->max_iter;
        s.status = TM_ERR_MAXITER;
        s.alpha_iter = -1;
    }
    TM_CUDA_CHECK(cudaMemcpyAsync(c.scal, h.data(), sizeof(CgScal) * nrhs, cudaMemcpyHostToDevice, st));
    TM_CUDA_CHECK(cudaMemsetAsync(c.active, 1, nrhs, st));
    TM_CUDA_CHECK(cudaMemsetAsync(c.tickets, 0, sizeof(unsigned int) * nrhs, st));
    // no stream synchronisation: a cudaMemcpyAsync from pageable host memory returns once the source has been staged, so `h`
    // may go out of scope here
    return TM_OK;
}

// b'' (stride pb) from the full-lattice source; t1, t2: scratch (stride pb)
static int prepare_rhs(const Geo& g, const void* gauge, int prec, int recon, const void* eta_full, void* b, void* t1, void* t2,
                       double kappa, double mu, int nrhs, cudaStream_t st, const void* link_cache = nullptr)
{
    const size_t pb = spinor_parity_bytes(g, prec);
    const char* eta_e = static_cast<const char*>(eta_full);
    const char* eta_o = eta_e + pb;
    const double a = 2.0 * kappa * mu, n = 1.0 / (1.0 + a * a);
    int rc;
    // t1 = R^-1 eta_o
    if ((rc = k_twist(g, prec, V_(t1, pb), V_(eta_o, 2 * pb), n, -a * n, nrhs, st)) != TM_OK) return rc;
    DslashParams p;
    p.gauge = gauge; p.nrhs = nrhs; p.active = nullptr; p.link_cache = link_cache;
    // t2 = b' = eta_e + kappa D_eo t1
    p.out = t2; p.in = t1; p.x = eta_e; p.out_parity = 0; p.dagger = 0;
    p.rhs_stride_out = pb; p.rhs_stride_in = pb; p.rhs_stride_x = 2 * pb;
    p.pq[0] = 1.0; p.pq[1] = 0.0; p.pq[2] = kappa; p.pq[3] = 0.0;
    if ((rc = launch_dslash(g, prec, recon, p, st)) != TM_OK) return rc;
    // t1 = R(-a)^-1 D^dag_oe b'
    p.out = t1; p.in = t2; p.x = nullptr; p.out_parity = 1; p.dagger = 1; p.rhs_stride_x = pb;
    kind_pq(TM_KIND_TWIST_INV, 1, kappa, mu, p.pq);
    if ((rc = launch_dslash(g, prec, recon, p, st)) != TM_OK) return rc;
    // b = R(-a) b' - kappa^2 D^dag_eo t1
    p.out = b; p.in = t1; p.x = t2; p.out_parity = 0;
    kind_pq(TM_KIND_XPAY_TWIST, 1, kappa, mu, p.pq);
    return launch_dslash(g, prec, recon, p, st);
}

// s_o = R^-1 eta_o + kappa R^-1 D_oe s_e   (all inside the full-lattice arrays, stride 2 pb)
static int reconstruct_odd(const Geo& g, const void* gauge, int prec, int recon, void* s_full, const void* eta_full, double kappa,
                           double mu, int nrhs, cudaStream_t st, const void* link_cache = nullptr)
{
    const size_t pb = spinor_parity_bytes(g, prec);
    const double a = 2.0 * kappa * mu, n = 1.0 / (1.0 + a * a);
    DslashParams p;
    p.gauge = gauge; p.nrhs = nrhs; p.active = nullptr; p.link_cache = link_cache;
    p.out = static_cast<char*>(s_full) + pb; p.in = s_full; p.x = static_cast<const char*>(eta_full) + pb;
    p.out_parity = 1; p.dagger = 0;
    p.rhs_stride_out = p.rhs_stride_in = p.rhs_stride_x = 2 * pb;
    p.pq[0] = n; p.pq[1] = -a * n; p.pq[2] = kappa * n; p.pq[3] = -kappa * a * n;
    return launch_dslash(g, prec, recon, p, st);
}

// The multi-rhs tile kernel (more than 6 right-hand sides, fp32 / fp16 storage) stages its links from a per-solve cache:
// one build (~0.3 ms at 32^3x64) serves the ~40-50 dslash launches of a truncated solve.
static inline bool lp_uses_link_cache(int prec, int nrhs) { return prec != 8 && nrhs > 6; }
static inline size_t dot_partial_bytes(const Geo& g, int nrhs) { return round256(sizeof(double) * (size_t)((g.Vh + 31) / 32) * nrhs); }

// Search-direction ring (tm_blas.cuh): used when its LP_RING_DEPTH - 1 extra stacks fit into TM_LP_RING_BYTES; otherwise the solution
// is updated inside the iteration (five vector passes per iteration instead of three + one pass per direction at a flush).
#ifndef TM_LP_RING_BYTES
#define TM_LP_RING_BYTES (size_t(16) << 30)
#endif
static inline int lp_ring_depth(const Geo& g, int prec, int nrhs)
{
    return (size_t)(LP_RING_DEPTH - 1) * round256(spinor_parity_bytes(g, prec) * nrhs) <= TM_LP_RING_BYTES ? LP_RING_DEPTH : 1;
}
static inline size_t lp_hist_bytes(int depth, int nrhs) { return round256(sizeof(double) * (size_t)(depth + 1) * nrhs); }

size_t cg_lp_workspace_bytes(const Geo& g, int prec, int nrhs)
{
    const int D = lp_ring_depth(g, prec, nrhs);
    const size_t stack = round256(spinor_parity_bytes(g, prec) * nrhs);
    return ctx_bytes(nrhs) + dot_partial_bytes(g, nrhs) + 6 * stack + (lp_uses_link_cache(prec, nrhs) ? link_cache_bytes(g, prec) : 0) +
           (D >= 2 ? (size_t)(D - 1) * stack + lp_hist_bytes(D, nrhs) : 0);
}

// truncated LP solve, batched
int cg_lp_truncated(const Geo& g, const void* gauge, int prec, int recon, void* s_full, const void* eta_full,
                    const tm_cg_params* prm, int nrhs, tm_cg_info* info, void* ws, size_t ws_bytes, cudaStream_t st)
{
    const size_t pb = spinor_parity_bytes(g, prec);
    Carver cv(ws, ws_bytes);
    BlasCtx c = carve_ctx(cv, nrhs);
    void* b = cv.take(pb * nrhs);
    void* r = cv.take(pb * nrhs);
    void* p = cv.take(pb * nrhs);
    void* Ap = cv.take(pb * nrhs);
    void* t1 = cv.take(2 * pb * nrhs); // t1, t2 contiguous (mdagm_apply tmp)
    void* t2 = static_cast<char*>(t1) + pb * nrhs;
    void* lc = lp_uses_link_cache(prec, nrhs) ? cv.take(link_cache_bytes(g, prec)) : nullptr;
    double* dotp = static_cast<double*>(cv.take(dot_partial_bytes(g, nrhs)));
    const int D = lp_ring_depth(g, prec, nrhs);
    void* ringbuf[LP_RING_DEPTH] = {p};
    double* hist = nullptr;
    if (D >= 2) {
        for (int j = 1; j < D; ++j) ringbuf[j] = cv.take(pb * nrhs);
        hist = static_cast<double*>(cv.take(sizeof(double) * (size_t)(D + 1) * nrhs));
    }
    if (!cv.ok()) return TM_ERR_LAYOUT;
    int rc;
    if ((rc = init_ctx(c, prm, nrhs, st)) != TM_OK) return rc;
    if (lc && (rc = link_cache_build(g, prec, recon, gauge, lc, st)) != TM_OK) return rc;
    if ((rc = prepare_rhs(g, gauge, prec, recon, eta_full, b, t1, t2, prm->kappa, prm->mu, nrhs, st, lc)) != TM_OK) return rc;
    if ((rc = k_norm2<FIN_INIT>(g, prec, V_(b, pb), c, nrhs, st)) != TM_OK) return rc;
    // r_0 = p_0 = b: iteration 0 reads both from b (k_cg_iter_fused), the stacks r and p are first written by it
    VecArg x = V_(s_full, 2 * pb); // s_e lives in the even block of s_full
    // x_0 = 0 is written by the vector kernel of iteration 0 (or by the first accumulation of the ring); only a solve without any
    // iteration and without a ring needs the memset
    if (prm->max_iter < 1 && D < 2) TM_CUDA_CHECK(cudaMemset2DAsync(s_full, 2 * pb, 0, pb, nrhs, st));
    // search direction p_j lives in b (j = 0) or in ring slot (j - 1) % D
    auto slot = [&](int j) -> void* { return j == 0 ? b : ringbuf[(j - 1) % D]; };
    int flushed = 0;      // x holds sum_{j < flushed} alpha_j p_j
    bool x_init = true;   // the first accumulation writes x instead of adding to it
    auto flush = [&](int upto) -> int {
        if (upto <= flushed && !x_init) return (int)TM_OK;
        XTerms t;
        t.n = 0;
        for (int j = flushed; j < upto; ++j, ++t.n) {
            t.p[t.n] = static_cast<const char*>(slot(j));
            t.stride[t.n] = pb;
            t.alpha[t.n] = hist + (size_t)(j % (D + 1)) * nrhs;
        }
        dim3 grid(blas_blocks(g.Vh), nrhs);
        const int init = x_init ? 1 : 0;
        const int rcf = by_prec(prec, [&](auto P) {
            accumulate_x_kernel<decltype(P)::value><<<grid, BLAS_THREADS, 0, st>>>(g.Vh, x, t, init);
            TM_LAUNCH_CHECK("accumulate_x_kernel");
            return (int)TM_OK;
        });
        flushed = upto > flushed ? upto : flushed;
        x_init = false;
        return rcf;
    };
    // one iteration: the fused operator launches, then either the classic x / p update or the ring update
    auto iterate = [&](int k) -> int {
        if (D < 2)
            return k_cg_iter_fused(g, gauge, prec, recon, x, V_(r, pb), V_(p, pb), V_(k == 0 ? b : r, pb), V_(k == 0 ? b : p, pb), t1, prm->kappa,
                                   prm->mu, c, dotp, nrhs, k, st, lc);
        void* pin = slot(k);
        void* pout = ringbuf[k % D];
        int rci = k_cg_iter_fused(g, gauge, prec, recon, x, V_(r, pb), V_(pout, pb), V_(k == 0 ? b : r, pb), V_(pin, pb), t1, prm->kappa, prm->mu, c,
                                  dotp, nrhs, k, st, lc, false);
        if (rci != TM_OK) return rci;
        // p_{k+1} overwrites p_{k+1-D}: flushing every LP_FLUSH_EVERY < D - 1 iterations keeps every unflushed direction alive
        if (k - flushed >= LP_FLUSH_EVERY && (rci = flush(k)) != TM_OK) return rci;
        dim3 grid(blas_blocks(g.Vh), nrhs);
        return by_prec(prec, [&](auto P) {
            update_p_hist_kernel<decltype(P)::value><<<grid, BLAS_THREADS, 0, st>>>(g.Vh, V_(pout, pb), V_(pin, pb), V_(r, pb), c, k,
                                                                                  hist + (size_t)(k % (D + 1)) * nrhs);
            TM_LAUNCH_CHECK("update_p_hist_kernel");
            return (int)TM_OK;
        });
    };
    int launched = 0; // iterations launched
    if (prm->check_every > 0) {
        // poll the device flags every `check_every` iterations (one stream synchronisation per poll)
        const int every = prm->check_every;
        unsigned char hact[TM_MAX_NRHS];
        for (int k = 0; k < prm->max_iter;) {
            for (int j = 0; j < every && k < prm->max_iter; ++j, ++k)
            {
                if ((rc = iterate(k)) != TM_OK) return rc;
                launched = k + 1;
            }
            TM_CUDA_CHECK(cudaMemcpyAsync(hact, c.active, nrhs, cudaMemcpyDeviceToHost, st));
            TM_CUDA_CHECK(cudaStreamSynchronize(st));
            bool any = false;
            for (int q = 0; q < nrhs; ++q) any |= hact[q] != 0;
            if (!any) break;
        }
    } else {
        // pipelined polling (check_every = 0): the flags of every iteration go to pinned host memory behind an event; the host
        // keeps one iteration queued ahead of the GPU and stops one iteration after the last right-hand side converged (the
        // extra iteration's kernels find no active rhs and exit).  The device never waits for the host.
        PollRing* ring = poll_ring();
        if (!ring) return TM_ERR_CUDA;
        for (int k = 0; k < prm->max_iter; ++k) {
            if ((rc = iterate(k)) != TM_OK) return rc;
            launched = k + 1;
            const int slot = k % PollRing::DEPTH;
            TM_CUDA_CHECK(cudaMemcpyAsync(ring->flags + slot * TM_MAX_NRHS, c.active, nrhs, cudaMemcpyDeviceToHost, st));
            TM_CUDA_CHECK(cudaEventRecord(ring->ev[slot], st));
            if (k >= 1) { // look at iteration k-1 while iteration k runs
                const int prev = (k - 1) % PollRing::DEPTH;
                TM_CUDA_CHECK(cudaEventSynchronize(ring->ev[prev]));
                bool any = false;
                for (int q = 0; q < nrhs; ++q) any |= ring->flags[prev * TM_MAX_NRHS + q] != 0;
                if (!any) break;
            }
        }
    }
    if (D >= 2 && (rc = flush(launched)) != TM_OK) return rc; // x = sum of the kept directions (zeros if nothing iterated)
    if ((rc = reconstruct_odd(g, gauge, prec, recon, s_full, eta_full, prm->kappa, prm->mu, nrhs, st, lc)) != TM_OK) return rc;
    // recomputed residual of the normal system, in the same storage/arithmetic: Ap = A x; Ap = b - Ap
    if (!prm->skip_true_resid) {
        if ((rc = mdagm_apply(g, gauge, prec, recon, Ap, pb, s_full, 2 * pb, t1, 0, prm->kappa, prm->mu, nrhs, nullptr, st, lc)) != TM_OK) return rc;
        if ((rc = k_axpby<1>(g, prec, prec, V_(Ap, pb), V_(b, pb), -1.0, 1.0, c, nrhs, st)) != TM_OK) return rc;
    }
    std::vector<CgScal> h(nrhs);
    TM_CUDA_CHECK(cudaMemcpyAsync(h.data(), c.scal, sizeof(CgScal) * nrhs, cudaMemcpyDeviceToHost, st));
    TM_CUDA_CHECK(cudaStreamSynchronize(st));
    int worst = TM_OK;
    for (int q = 0; q < nrhs; ++q) {
        info[q].iters = h[q].iter;
        info[q].status = h[q].status;
        info[q].reliable_updates = 0;
        info[q].iterated_resid = h[q].b2 > 0 ? std::sqrt(h[q].rr / h[q].b2) : 0.0;
        info[q].true_resid = prm->skip_true_resid ? -1.0 : (h[q].b2 > 0 ? std::sqrt(h[q].aux / h[q].b2) : 0.0);
        if (h[q].b2 == 0.0) info[q].status = TM_OK;
        if (info[q].status == TM_ERR_MAXITER && prm->tol == 0.0) info[q].status = TM_OK; // fixed-iteration truncation
        if (info[q].status != TM_OK && (worst == TM_OK || info[q].status == TM_ERR_BREAKDOWN)) worst = info[q].status;
    }
    return worst;
}

} // namespace tmk

namespace tmk {

size_t cg_hp_workspace_bytes(const Geo& g, int prec_hp, int prec_lp)
{
    return ctx_bytes(1) + 4 * round256(spinor_parity_bytes(g, prec_hp)) + 6 * round256(spinor_parity_bytes(g, prec_lp));
}

static int read_scal(const BlasCtx& c, CgScal* h, cudaStream_t st)
{
    TM_CUDA_CHECK(cudaMemcpyAsync(h, c.scal, sizeof(CgScal), cudaMemcpyDeviceToHost, st));
    TM_CUDA_CHECK(cudaStreamSynchronize(st));
    return TM_OK;
}

static int write_scal(const BlasCtx& c, const CgScal* h, unsigned char active, cudaStream_t st)
{
    TM_CUDA_CHECK(cudaMemcpyAsync(c.scal, h, sizeof(CgScal), cudaMemcpyHostToDevice, st));
    TM_CUDA_CHECK(cudaMemsetAsync(c.active, active, 1, st));
    TM_CUDA_CHECK(cudaStreamSynchronize(st));
    return TM_OK;
}

// mixed-precision solve of ONE right-hand side: CG iterations in prec_lp, reliable updates in prec_hp
// (reading 10).  eta_full / s_full are packed at prec_hp.
int cg_hp_mixed(const Geo& g, const void* gauge_hp, int prec_hp, const void* gauge_lp, int prec_lp, int recon, void* s_full,
                const void* eta_full, const tm_cg_params* prm, tm_cg_info* info, void* ws, size_t ws_bytes, cudaStream_t st)
{
    const size_t pbh = spinor_parity_bytes(g, prec_hp), pbl = spinor_parity_bytes(g, prec_lp);
    Carver cv(ws, ws_bytes);
    BlasCtx c = carve_ctx(cv, 1);
    void* b = cv.take(pbh);
    void* rh = cv.take(pbh);
    void* th = cv.take(2 * pbh);
    void* r = cv.take(pbl);
    void* p = cv.take(pbl);
    void* Ap = cv.take(pbl);
    void* xl = cv.take(pbl);
    void* tl = cv.take(2 * pbl);
    if (!cv.ok()) return TM_ERR_LAYOUT;
    const double kappa = prm->kappa, mu = prm->mu;
    const double delta = prm->reliable_delta > 0 ? prm->reliable_delta : 0.1;
    int rc;
    if ((rc = init_ctx(c, prm, 1, st)) != TM_OK) return rc;
    if ((rc = prepare_rhs(g, gauge_hp, prec_hp, recon, eta_full, b, th, static_cast<char*>(th) + pbh, kappa, mu, 1, st)) != TM_OK) return rc;
    if ((rc = k_norm2<FIN_INIT>(g, prec_hp, V_(b, pbh), c, 1, st)) != TM_OK) return rc;
    if ((rc = k_convert(g, prec_lp, prec_hp, V_(r, pbl), V_(p, pbl), V_(b, pbh), 1, st)) != TM_OK) return rc;
    TM_CUDA_CHECK(cudaMemsetAsync(s_full, 0, pbh, st)); // x_hp = s_e = 0
    TM_CUDA_CHECK(cudaMemsetAsync(xl, 0, pbl, st));
    CgScal h;
    if ((rc = read_scal(c, &h, st)) != TM_OK) return rc;
    const double b2 = h.b2;
    info->iters = 0; info->reliable_updates = 0; info->status = TM_OK; info->iterated_resid = 0; info->true_resid = 0;
    if (!(b2 > 0.0)) {
        TM_CUDA_CHECK(cudaMemsetAsync(s_full, 0, 2 * pbh, st));
        return reconstruct_odd(g, gauge_hp, prec_hp, recon, s_full, eta_full, kappa, mu, 1, st);
    }
    // the LP iteration never decides convergence on its own: tol2 = 0 on the device, the host decides
    h.tol2 = 0.0;
    if ((rc = write_scal(c, &h, 1, st)) != TM_OK) return rc;
    double rr_prev = h.rr, rr_max = h.rr, rr_true = h.rr;
    const double target2 = prm->tol * prm->tol * b2;
    int status = TM_ERR_MAXITER;
    bool x_dirty = false;
    int k = 0;
    while (k < prm->max_iter) {
        if ((rc = k_cg_iter(g, gauge_lp, prec_lp, recon, V_(xl, pbl), V_(r, pbl), V_(p, pbl), V_(Ap, pbl), tl, kappa, mu, c, 1, false,
                            st)) != TM_OK)
            return rc;
        ++k;
        x_dirty = true;
        if ((rc = read_scal(c, &h, st)) != TM_OK) return rc;
        if (h.status == TM_ERR_BREAKDOWN) {
            // keep what the iterations since the last reliable update have gained: x_hp += x_lp before the odd sites are rebuilt
            if (x_dirty && (rc = k_axpby<0>(g, prec_hp, prec_lp, V_(s_full, 2 * pbh), V_(xl, pbl), 1.0, 1.0, c, 1, st)) != TM_OK) return rc;
            x_dirty = false;
            status = TM_ERR_BREAKDOWN;
            break;
        }
        const double rr = h.rr;
        if (rr > rr_max) rr_max = rr;
        const bool want = (rr < delta * delta * rr_max) || (rr <= target2) || (k == prm->max_iter);
        if (want) {
            // x_hp += x_lp; x_lp = 0; r_hp = b - A_hp x_hp
            if ((rc = k_axpby<0>(g, prec_hp, prec_lp, V_(s_full, 2 * pbh), V_(xl, pbl), 1.0, 1.0, c, 1, st)) != TM_OK) return rc;
            TM_CUDA_CHECK(cudaMemsetAsync(xl, 0, pbl, st));
            x_dirty = false;
            if ((rc = mdagm_apply(g, gauge_hp, prec_hp, recon, rh, pbh, s_full, 2 * pbh, th, 0, kappa, mu, 1, nullptr, st)) != TM_OK) return rc;
            if ((rc = k_axpby<1>(g, prec_hp, prec_hp, V_(rh, pbh), V_(b, pbh), -1.0, 1.0, c, 1, st)) != TM_OK) return rc;
            if ((rc = k_convert(g, prec_lp, prec_hp, V_(r, pbl), V_((void*)nullptr, 0), V_(rh, pbh), 1, st)) != TM_OK) return rc;
            if ((rc = read_scal(c, &h, st)) != TM_OK) return rc;
            rr_true = h.aux;
            info->reliable_updates += 1;
            info->iterated_resid = std::sqrt(rr / b2);
            if (rr_true <= target2) { status = TM_OK; break; }
            h.rr = rr_true;
            h.beta = rr_true / rr_prev;
            h.status = TM_ERR_MAXITER;
            if ((rc = write_scal(c, &h, 1, st)) != TM_OK) return rc;
            rr_max = rr_true;
            rr_prev = rr_true;
        } else {
            rr_prev = rr;
            info->iterated_resid = std::sqrt(rr / b2);
        }
        if (k < prm->max_iter)
            if ((rc = k_update_p(g, prec_lp, V_(p, pbl), V_(r, pbl), c, 1, st)) != TM_OK) return rc;
    }
    info->iters = k;
    info->status = status;
    info->true_resid = std::sqrt(rr_true / b2);
    if ((rc = reconstruct_odd(g, gauge_hp, prec_hp, recon, s_full, eta_full, kappa, mu, 1, st)) != TM_OK) return rc;
    TM_CUDA_CHECK(cudaStreamSynchronize(st));
    return status;
}

// aux of context entry 2 rhs (+ the parity offset already applied to c.scal) = sum of the per-warp partials, fixed order
__global__ void __launch_bounds__(BLAS_THREADS) dot_finalize_strided_kernel(const double* partial, int ngroups, BlasCtx c)
{
    const int rhs = blockIdx.x;
    double v = 0.0;
    const double* p = partial + (size_t)rhs * ngroups;
    for (int g = threadIdx.x; g < ngroups; g += BLAS_THREADS) v += p[g];
    const double tot = block_sum(v);
    if (threadIdx.x == 0) c.scal[2 * rhs].aux = tot;
}

// ---- HP by defect correction, batched (TM_CG_HP_DEFECT) ---------------------------------------------------------------
// The alternative SURVEY.md 8(c-2) reading 10 names: outer residual and solution in the HP precision, inner solves by the
// BATCHED truncated LP solver (every gauge load shared by all right-hand sides), restarted each cycle:
//     s = 0, r = eta;  repeat: e = LP-solve(M e = r) to relative tolerance `reliable_delta`;  s += e;  r = eta - M s (HP)
// until |eta - M s| <= tol |eta| for every right-hand side (the residual of the FULL system, both parities).
int full_operator(const Geo& g, const void* gauge, int prec, int recon, void* out_full, const void* in_full, double kappa, double mu,
                  int dagger, int nrhs, cudaStream_t st);

size_t cg_defect_workspace_bytes(const Geo& g, int prec_hp, int prec_lp, int nrhs)
{
    return ctx_bytes(2 * nrhs) + round256(2 * spinor_parity_bytes(g, prec_hp) * nrhs) + 2 * round256(2 * spinor_parity_bytes(g, prec_lp) * nrhs) +
           cg_lp_workspace_bytes(g, prec_lp, nrhs) + 2 * dot_partial_bytes(g, nrhs) + round256(sizeof(double) * nrhs);
}

int cg_hp_defect(const Geo& g, const void* gauge_hp, int prec_hp, const void* gauge_lp, int prec_lp, int recon, void* s_full,
                 const void* eta_full, const tm_cg_params* prm, int nrhs, tm_cg_info* info, void* ws, size_t ws_bytes, cudaStream_t st)
{
    const size_t pbh = spinor_parity_bytes(g, prec_hp), pbl = spinor_parity_bytes(g, prec_lp);
    const int nv = 2 * nrhs; // full-lattice arrays [rhs][parity] seen as nv one-parity vectors
    Carver cv(ws, ws_bytes);
    BlasCtx c = carve_ctx(cv, nv);
    void* R = cv.take(2 * pbh * nrhs);
    void* r_lp = cv.take(2 * pbl * nrhs);
    void* e_lp = cv.take(2 * pbl * nrhs);
    const size_t lpb = cg_lp_workspace_bytes(g, prec_lp, nrhs);
    void* lpws = cv.take(lpb);
    double* dotp[2] = {static_cast<double*>(cv.take(dot_partial_bytes(g, nrhs))), static_cast<double*>(cv.take(dot_partial_bytes(g, nrhs)))};
    double* ones = static_cast<double*>(cv.take(sizeof(double) * nrhs));
    if (!cv.ok()) return TM_ERR_LAYOUT;
    int rc;
    {
        const std::vector<double> one(nrhs, 1.0);
        TM_CUDA_CHECK(cudaMemcpyAsync(ones, one.data(), sizeof(double) * nrhs, cudaMemcpyHostToDevice, st));
        TM_CUDA_CHECK(cudaStreamSynchronize(st));
    }
    tm_cg_params zero = *prm;
    if ((rc = init_ctx(c, &zero, nv, st)) != TM_OK) return rc;
    std::vector<CgScal> h(nv);
    auto read_aux = [&](std::vector<double>& out) -> int {
        TM_CUDA_CHECK(cudaMemcpyAsync(h.data(), c.scal, sizeof(CgScal) * nv, cudaMemcpyDeviceToHost, st));
        TM_CUDA_CHECK(cudaStreamSynchronize(st));
        for (int q = 0; q < nrhs; ++q) out[q] = h[2 * q].aux + h[2 * q + 1].aux;
        return TM_OK;
    };
    std::vector<double> b2(nrhs), r2(nrhs);
    if ((rc = k_norm2<FIN_AUX>(g, prec_hp, V_(eta_full, pbh), c, nv, st)) != TM_OK) return rc;
    if ((rc = read_aux(b2)) != TM_OK) return rc;
    TM_CUDA_CHECK(cudaMemsetAsync(s_full, 0, 2 * pbh * nrhs, st));
    TM_CUDA_CHECK(cudaMemcpyAsync(R, eta_full, 2 * pbh * nrhs, cudaMemcpyDeviceToDevice, st));
    r2 = b2;
    tm_cg_params inner = *prm;
    inner.mode = TM_CG_LP_TRUNCATED;
    inner.tol = (prm->reliable_delta > 0 && prm->reliable_delta < 1) ? prm->reliable_delta : 1e-3;
    inner.skip_true_resid = 1;
    inner.check_every = 0;
    std::vector<tm_cg_info> iinfo(nrhs);
    for (int q = 0; q < nrhs; ++q) {
        info[q].iters = 0;
        info[q].reliable_updates = 0;
        info[q].status = TM_ERR_MAXITER;
    }
    int total = 0;
    bool done = false;
    auto converged = [&]() {
        bool all = true;
        for (int q = 0; q < nrhs; ++q) {
            const bool ok = b2[q] == 0.0 || r2[q] <= prm->tol * prm->tol * b2[q];
            if (ok && info[q].status == TM_ERR_MAXITER) info[q].status = TM_OK;
            all = all && ok;
        }
        return all;
    };
    done = converged();
    int worst = TM_OK;
    for (int cycle = 0; !done && total < prm->max_iter && cycle < 64; ++cycle) {
        inner.max_iter = prm->max_iter - total;
        // the last cycle only has to close the remaining gap: relax the inner tolerance to 0.3 tol / (worst current residual)
        double worst_rel = 0.0;
        for (int q = 0; q < nrhs; ++q)
            if (b2[q] > 0) worst_rel = std::max(worst_rel, std::sqrt(r2[q] / b2[q]));
        const double base_tol = (prm->reliable_delta > 0 && prm->reliable_delta < 1) ? prm->reliable_delta : 1e-3;
        inner.tol = worst_rel > 0 ? std::min(0.5, std::max(base_tol, 0.3 * prm->tol / worst_rel)) : base_tol;
        if ((rc = k_convert(g, prec_lp, prec_hp, V_(r_lp, pbl), VecArg{nullptr, 0}, V_(R, pbh), nv, st)) != TM_OK) return rc;
        rc = cg_lp_truncated(g, gauge_lp, prec_lp, recon, e_lp, r_lp, &inner, nrhs, iinfo.data(), lpws, lpb, st);
        if (rc == TM_ERR_CUDA || rc == TM_ERR_LAYOUT) return rc;
        if (rc == TM_ERR_BREAKDOWN) worst = rc;
        int it = 0;
        for (int q = 0; q < nrhs; ++q) {
            if (info[q].status == TM_ERR_MAXITER) { // still being refined: count its inner iterations and this cycle
                info[q].iters += iinfo[q].iters;
                info[q].reliable_updates += 1;
            }
            it = iinfo[q].iters > it ? iinfo[q].iters : it;
        }
        total += it > 0 ? it : 1;
        // s += e (HP += LP), then R = eta - M s in HP: the subtraction and |R|^2 ride on the epilogue of the two dslash launches
        // (fused_axpy with coefficient 1, per-warp fp64 partials), so eta, M s and R are not streamed a second time
        if ((rc = k_axpby<0>(g, prec_hp, prec_lp, V_(s_full, pbh), V_(e_lp, pbl), 1.0, 1.0, c, nv, st)) != TM_OK) return rc;
        for (int parity = 0; parity < 2; ++parity) {
            DslashParams dp;
            dp.gauge = gauge_hp; dp.nrhs = nrhs; dp.active = nullptr; dp.dagger = 0;
            dp.out = static_cast<char*>(R) + parity * pbh;
            dp.in = static_cast<const char*>(s_full) + (1 - parity) * pbh;
            dp.x = static_cast<const char*>(s_full) + parity * pbh;
            dp.out_parity = parity;
            dp.rhs_stride_out = dp.rhs_stride_in = dp.rhs_stride_x = 2 * pbh;
            dp.pq[0] = 1.0; dp.pq[1] = 2.0 * prm->kappa * prm->mu; dp.pq[2] = -prm->kappa; dp.pq[3] = 0.0;
            dp.axpy_y = static_cast<const char*>(eta_full) + parity * pbh;
            dp.axpy_y_stride = 2 * pbh;
            dp.axpy_coef = ones;
            dp.axpy_coef_stride = sizeof(double);
            dp.dot_partial = dotp[parity];
            if ((rc = launch_dslash(g, prec_hp, recon, dp, st)) != TM_OK) return rc;
            // vector index of (rhs q, parity) in the context is 2 q + parity: finalize with a strided view of the context
            BlasCtx cp = c;
            cp.scal = c.scal + parity;
            cp.active = c.active + parity;
            dot_finalize_strided_kernel<<<nrhs, BLAS_THREADS, 0, st>>>(dotp[parity], (g.Vh + 31) / 32, cp);
            TM_LAUNCH_CHECK("dot_finalize_strided_kernel");
        }
        if ((rc = read_aux(r2)) != TM_OK) return rc;
        done = converged();
    }
    for (int q = 0; q < nrhs; ++q) {
        const double rel = b2[q] > 0 ? std::sqrt(r2[q] / b2[q]) : 0.0;
        info[q].iterated_resid = rel;
        info[q].true_resid = rel;
        if (info[q].status != TM_OK && worst == TM_OK) worst = info[q].status;
    }
    return worst;
}

} // namespace tmk

using namespace tmk;

extern "C" size_t tm_cg_workspace_bytes(const tm_lattice* L, int prec_hp, int prec_lp, int mode, int nrhs)
{
    if (!L || !valid_prec(prec_lp) || nrhs < 1 || nrhs > TM_MAX_NRHS) return 0;
    if (mode == TM_CG_LP_TRUNCATED) return cg_lp_workspace_bytes(L->g, prec_lp, nrhs);
    if (!valid_prec(prec_hp)) return 0;
    if (mode == TM_CG_HP_DEFECT) return cg_defect_workspace_bytes(L->g, prec_hp, prec_lp, nrhs);
    return cg_hp_workspace_bytes(L->g, prec_hp, prec_lp);
}

extern "C" int tm_cg_multi(const tm_lattice* L, const void* gauge_hp, int prec_hp, const void* gauge_lp, int prec_lp, int recon,
                           void* s_full, const void* eta_full, const tm_cg_params* p, int nrhs, tm_cg_info* info, void* workspace,
                           size_t workspace_bytes, void* stream)
{
    if (!L || !gauge_lp || !s_full || !eta_full || !p || !info || !workspace) return TM_ERR_ARG;
    if (!valid_prec(prec_lp) || !valid_recon(recon) || nrhs < 1 || nrhs > TM_MAX_NRHS || p->max_iter < 0 || p->tol < 0) return TM_ERR_ARG;
    if (!aligned256(gauge_lp) || !aligned256(s_full) || !aligned256(eta_full) || !aligned256(workspace)) return TM_ERR_LAYOUT;
    if (workspace_bytes < tm_cg_workspace_bytes(L, prec_hp, prec_lp, p->mode, nrhs)) return TM_ERR_LAYOUT;
    cudaStream_t st = (cudaStream_t)stream;
    if (p->mode == TM_CG_LP_TRUNCATED)
        return cg_lp_truncated(L->g, gauge_lp, prec_lp, recon, s_full, eta_full, p, nrhs, info, workspace, workspace_bytes, st);
    if ((p->mode != TM_CG_HP_MIXED && p->mode != TM_CG_HP_DEFECT) || !gauge_hp || !valid_prec(prec_hp) || !aligned256(gauge_hp)) return TM_ERR_ARG;
    if (p->mode == TM_CG_HP_DEFECT)
        return cg_hp_defect(L->g, gauge_hp, prec_hp, gauge_lp, prec_lp, recon, s_full, eta_full, p, nrhs, info, workspace, workspace_bytes, st);
    // HP_MIXED: right-hand sides are solved one after the other (reliable-update decisions are per solve)
    const size_t fb = 2 * spinor_parity_bytes(L->g, prec_hp);
    int worst = TM_OK;
    for (int q = 0; q < nrhs; ++q) {
        const int rc = cg_hp_mixed(L->g, gauge_hp, prec_hp, gauge_lp, prec_lp, recon, static_cast<char*>(s_full) + q * fb,
                                   static_cast<const char*>(eta_full) + q * fb, p, info + q, workspace, workspace_bytes, st);
        if (rc == TM_ERR_CUDA || rc == TM_ERR_LAYOUT) return rc;
        if (rc != TM_OK && (worst == TM_OK || rc == TM_ERR_BREAKDOWN)) worst = rc;
    }
    return worst;
}

extern "C" int tm_cg(const tm_lattice* L, const void* gauge_hp, int prec_hp, const void* gauge_lp, int prec_lp, int recon,
                     void* s_full, const void* eta_full, const tm_cg_params* p, tm_cg_info* info, void* workspace,
                     size_t workspace_bytes, void* stream)
{
    return tm_cg_multi(L, gauge_hp, prec_hp, gauge_lp, prec_lp, recon, s_full, eta_full, p, 1, info, workspace, workspace_bytes, stream);
}

extern "C" size_t tm_tsm_workspace_bytes(const tm_lattice* L, int prec_lp, int nrhs)
{
    if (!L || !valid_prec(prec_lp) || nrhs < 1 || nrhs > TM_MAX_NRHS) return 0;
    const size_t fb = 2 * spinor_parity_bytes(L->g, prec_lp) * nrhs;
    return round256((size_t)L->V * 12 * nrhs) + 2 * round256(fb) + cg_lp_workspace_bytes(L->g, prec_lp, nrhs) +
           loop_workspace_bytes(L->g, nrhs) + round256((size_t)nrhs * 16 * L->g.T * 2 * sizeof(double));
}

static int tsm_batch_host(const tm_lattice* L, const void* gauge_lp, int prec_lp, int recon, const unsigned char* codes_host,
                          int bytes_per_site, const tm_cg_params* p, int nrhs, tm_cg_info* info, double* loops_host, void* workspace,
                          size_t workspace_bytes, void* stream)
{
    if (!L || !gauge_lp || !codes_host || !p || !info || !loops_host || !workspace) return TM_ERR_ARG;
    if (!valid_prec(prec_lp) || !valid_recon(recon) || nrhs < 1 || nrhs > TM_MAX_NRHS) return TM_ERR_ARG;
    if (!aligned256(gauge_lp) || !aligned256(workspace)) return TM_ERR_LAYOUT;
    if (workspace_bytes < tm_tsm_workspace_bytes(L, prec_lp, nrhs)) return TM_ERR_LAYOUT;
    cudaStream_t st = (cudaStream_t)stream;
    const Geo& g = L->g;
    const size_t fb = 2 * spinor_parity_bytes(g, prec_lp) * nrhs;
    Carver cv(workspace, workspace_bytes);
    unsigned char* codes = static_cast<unsigned char*>(cv.take((size_t)L->V * 12 * nrhs));
    void* eta = cv.take(fb);
    void* s = cv.take(fb);
    const size_t cgb = cg_lp_workspace_bytes(g, prec_lp, nrhs);
    void* cgws = cv.take(cgb);
    void* lws = cv.take(loop_workspace_bytes(g, nrhs));
    const size_t lb = (size_t)nrhs * 16 * g.T * 2 * sizeof(double);
    double* loops = static_cast<double*>(cv.take(lb));
    if (!cv.ok()) return TM_ERR_LAYOUT;
    TM_CUDA_CHECK(cudaMemcpyAsync(codes, codes_host, (size_t)L->V * bytes_per_site * nrhs, cudaMemcpyHostToDevice, st));
    int rc = spinor_pack_any(g, L->V, prec_lp, bytes_per_site == 3 ? 3 : 2, nullptr, nullptr, codes, eta, nrhs, st);
    if (rc != TM_OK) return rc;
    tm_cg_params q = *p;
    q.mode = TM_CG_LP_TRUNCATED;
    const int rc_cg = cg_lp_truncated(g, gauge_lp, prec_lp, recon, s, eta, &q, nrhs, info, cgws, cgb, st);
    if (rc_cg == TM_ERR_CUDA || rc_cg == TM_ERR_LAYOUT) return rc_cg;
    if ((rc = loop_contract(g, eta, s, prec_lp, nrhs, loops, lws, st)) != TM_OK) return rc;
    TM_CUDA_CHECK(cudaMemcpyAsync(loops_host, loops, lb, cudaMemcpyDeviceToHost, st));
    TM_CUDA_CHECK(cudaStreamSynchronize(st));
    return rc_cg;
}

extern "C" int tm_tsm_batch_host(const tm_lattice* L, const void* gauge_lp, int prec_lp, int recon, const unsigned char* codes_host,
                                 const tm_cg_params* p, int nrhs, tm_cg_info* info, double* loops_host, void* workspace,
                                 size_t workspace_bytes, void* stream)
{
    return tsm_batch_host(L, gauge_lp, prec_lp, recon, codes_host, 12, p, nrhs, info, loops_host, workspace, workspace_bytes, stream);
}

extern "C" int tm_tsm_batch_host_bits(const tm_lattice* L, const void* gauge_lp, int prec_lp, int recon, const unsigned char* codes3_host,
                                      const tm_cg_params* p, int nrhs, tm_cg_info* info, double* loops_host, void* workspace,
                                      size_t workspace_bytes, void* stream)
{
    return tsm_batch_host(L, gauge_lp, prec_lp, recon, codes3_host, 3, p, nrhs, info, loops_host, workspace, workspace_bytes, stream);
}
