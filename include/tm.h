/*
 * tm.h -- C ABI of the B200-native twisted-mass dslash / MdagM / CG / loop library (libtm_b200.so).
 *
 * Hot path of arxiv/paper_1309_2256 ("Evaluation of disconnected quark loops for hadron structure using GPUs").
 * Citations are PAPER.md:<line> plus section / equation.  Readings of the paper are listed in DESIGN.md.
 *
 * General rules
 *  - Plain C types only.  `stream` arguments are a cudaStream_t passed as void* (NULL = legacy default stream).
 *  - OWNERSHIP: the caller owns all device memory.  The library never allocates device memory; workspaces are
 *    passed in, sized by the tm_*_bytes() queries.  Pointers are borrowed until the stream work completes.
 *    Every device buffer must be 256-byte aligned; the one-parity spinor arguments of tm_dslash* / tm_MdagM may also be the
 *    even / odd block of a full-lattice buffer (16-byte alignment suffices there).  "device" / "host" is stated per argument.
 *  - ERRORS: every entry point returns int: TM_OK (0) or a negative tm_status.  No exceptions, no exit().
 *    Calls are asynchronous on `stream` unless they fill host structs (tm_cg*, tm_tsm_batch_host: documented).
 *  - There is no CPU fallback: without a CUDA device every compute call returns TM_ERR_CUDA.
 *
 * Conventions (identical to the oracle's, DESIGN.md section "Readings")
 *  - Lattice X x Y x Z x T, all even and >= 4; site = x + X*(y + Y*(z + Z*t)); mu = 0..3 = x,y,z,t;
 *    parity = (x+y+z+t)&1, even = 0.  Periodic in space, time antiperiodic if the lattice was created so.
 *  - Canonical fields (fp64, complex interleaved): gauge U[site][mu][row][col][re,im],
 *    spinor psi[site][spin][colour][re,im].
 *  - Dslash = positive hopping sum
 *      (Dslash psi)(x) = sum_mu (1-g_mu) s_mu(x) U_mu(x) psi(x+mu) + (1+g_mu) s_mu(x-mu) U_mu(x-mu)^dag psi(x-mu),
 *    M(kappa,mu) = 1 + i a g5 - kappa Dslash, a = 2 kappa mu  (PAPER.md:162 Eq. 16 B, H; :367 Eq. A1).
 *    Chiral gamma basis: g_k = [[0,-i s_k],[i s_k,0]], g_4 = [[0,1],[1,0]], g5 = diag(1,1,-1,-1).
 *  - Packed device layout: per parity, checkerboard index cb = site>>1;
 *    structure of arrays in 16-byte chunks [chunk][cb]; fp16 spinors carry one fp32 norm per site.
 */
#ifndef TM_B200_H
#define TM_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TM_VERSION 100

typedef struct tm_lattice tm_lattice; /* opaque host-side geometry descriptor */

typedef enum { TM_PREC_F64 = 8, TM_PREC_F32 = 4, TM_PREC_F16 = 2 } tm_prec;   /* storage bytes per real */
/* reals stored per link.  The *_FIX16 codes (reals + 100) select 16-bit FIXED-POINT link words for
 * TM_PREC_F16 fields (Fig. 4 names only "16-bit (half)" precision; the fixed-point word is SURVEY.md 8(f) NEXT-4's variant of it, reading 32): every stored real is
 * the offset-binary word q + 32768, q = rint(32767 u) in [-32767, 32767], value q / 32767 (+-1 exact, absolute error <= 1.6e-5
 * against up to 2.4e-4 for binary16 entries near 1); same bytes and chunk layout as the binary16 links.  With TM_PREC_F64 /
 * TM_PREC_F32 the flag is ignored (the field is the plain 18 / 12-real one), so one `recon` serves a mixed-precision solve.
 * The *_TG codes (reals + 200) DECLARE a field in temporal gauge: the temporal links of the slices t < T-1 are exactly the unit matrix (not in
 * the paper; reading 33).  tm_gauge_pack verifies the declaration (TM_ERR_NOT_TGAUGE otherwise) and stores the field like the plain
 * 18 / 12-real one -- unit links included, so a kernel that ignores the declaration is still correct.  The single-right-hand-side fp32 / fp16
 * hopping-term kernels honour it: temporal hops that do not wrap around load no link and multiply by none (25 % fewer link bytes, 144
 * fewer multiply-adds per site); every other kernel treats the code as the plain one.
 * HAZARD: the declaration travels in the `recon` ARGUMENT of each call, not in the packed buffer (same bytes and size as the plain code), so
 * only the pack call can verify it.  Passing a *_TG code to tm_dslash / tm_MdagM / tm_cg* / tm_M for a buffer that was packed under the plain
 * code (or from a field that is not in temporal gauge) silently skips non-unit temporal links and returns wrong results with TM_OK.
 * Use a *_TG code only with the buffer the pack call accepted under that code. */
typedef enum { TM_RECON_18 = 18, TM_RECON_12 = 12, TM_RECON_8 = 8, TM_RECON_18_FIX16 = 118, TM_RECON_12_FIX16 = 112,
               TM_RECON_18_TG = 218, TM_RECON_12_TG = 212 } tm_recon;
typedef enum { TM_KIND_PLAIN = 0, TM_KIND_TWIST_INV = 1, TM_KIND_XPAY_TWIST = 2 } tm_dslash_kind;
typedef enum { TM_CG_HP_MIXED = 0, TM_CG_LP_TRUNCATED = 1, TM_CG_HP_DEFECT = 2 } tm_cg_mode;

typedef enum {
    TM_OK = 0,
    TM_ERR_ARG = -1,       /* null pointer, bad enum, aliasing out == in, nrhs out of range */
    TM_ERR_LAYOUT = -2,    /* dims odd or < 4, misaligned buffer, workspace too small */
    TM_ERR_NOT_SU3 = -3,   /* tm_gauge_pack with recon 12: a link is farther than su3_tol from SU(3) */
    TM_ERR_CUDA = -4,      /* CUDA runtime error (no device, launch failure); tm_last_cuda_error() has the text */
    TM_ERR_BREAKDOWN = -5, /* CG: <p,Ap> <= 0 or NaN */
    TM_ERR_MAXITER = -6,   /* CG: max_iter reached before tol (solution still returned) */
    TM_ERR_RECON8 = -7,    /* tm_gauge_pack with recon 8: a link has |U00|^2 + |U01|^2 < 1e-6 (|U02| = 1), where the 8-real chart is singular */
    TM_ERR_NOT_TGAUGE = -8, /* tm_gauge_pack with a *_TG code: a temporal link of a slice t < T-1 is not exactly the unit matrix */
    TM_ERR_STATIC_LIMIT = -9 /* tm_loop_contract_static: the call needs more than TM_LOOP_STATIC_BYTES of scratch; use tm_loop_contract */
} tm_status;

#define TM_MAX_NRHS 16

int tm_version(void);
const char* tm_strerror(int status);
const char* tm_last_cuda_error(void);

/* ---- geometry ------------------------------------------------------------------------------------------ */
/* dims = {X,Y,Z,T}.  antiperiodic_t != 0: hops across t = T-1 <-> 0 carry -1 (BASELINE.json configs[0]). */
int tm_lattice_create(tm_lattice** L, const int dims[4], int antiperiodic_t);
void tm_lattice_destroy(tm_lattice* L);

/* ---- sizes --------------------------------------------------------------------------------------------- */
size_t tm_gauge_bytes(const tm_lattice* L, int prec, int recon);
/* full != 0: both parities ([even block][odd block]); else one parity.  nrhs fields are stacked [rhs][...]. */
size_t tm_spinor_bytes(const tm_lattice* L, int prec, int full, int nrhs);

/* ---- a0: gauge pack (links stored with 12 parameters and rebuilt on the fly) ------------- */
/* U_canonical: DEVICE, fp64 canonical, 4*V*18 doubles.  packed_out: DEVICE, tm_gauge_bytes().
 * recon 12 keeps rows 0,1 (row 2 = conj(row0 x row1) is rebuilt in the kernels; the antiperiodic sign is NOT
 * folded into stored links).  With recon 12, returns TM_ERR_NOT_SU3 if max |U U^dag - 1|, |row2 - conj(r0 x r1)|
 * exceeds su3_tol (this check synchronises the stream); su3_tol <= 0 skips the check.
 * recon 8 ("8-parameter reconstruction"): of V = U P, V_ij = U_{i,(j+2)%3} (columns shifted cyclically; still SU(3)) the
 * numbers V01, V02, V10 and arg(V00)/pi, arg(V20)/pi are stored; the kernels rebuild V from unitarity (two square roots, two sincospi,
 * one reciprocal of r = |V01|^2 + |V02|^2 = |U00|^2 + |U01|^2: errors grow like 1/r; reading 31) and undo the shift by
 * renaming.  The shift puts the chart's singular set at |U02| = 1 instead of the unit link, so free fields and temporal-gauge
 * fields pack.  Same SU(3) check as recon 12; a field with a link of r < 1e-6 is refused with TM_ERR_RECON8 (this check always
 * synchronises the stream). */
int tm_gauge_pack(const tm_lattice* L, const double* U_canonical, int prec, int recon, void* packed_out,
                  double su3_tol, void* stream);

/* Synthetic SU(3) gauge field made on the device (PAPER.md:250 has sources, inversions and contractions on the
 * GPUs -- the paper READS its gauge field from an ensemble, this call exists for the synthetic stand-in of DESIGN.md section 4): link
 * (site, mu) = Gram-Schmidt SU(3) projection of w 1 + eps G, G complex Gaussian from the counter-based splitmix64 hash of
 * (seed, 4 site + mu, draw), the generator of tm_inputs restated.  U_canonical_out: DEVICE fp64 [V][4][3][3][re,im] (the layout
 * tm_gauge_pack reads).  The hashes equal the host generator's bit for bit; log / cos / sin are the device's, so every real of a link
 * agrees with the host field to 1e-13 (measured on 32^3 x 64: median 1.1e-16, 99.99 % of the links below 2e-15, worst of 8.4 M links
 * 1.8e-14 where a normalisation amplifies the last-bit differences) and |U U^dag - 1| < 5e-14 -- not bit-identical.  Asynchronous on `stream`. */
int tm_gauge_synthetic(const tm_lattice* L, unsigned long long seed, double w, double eps, double* U_canonical_out, void* stream);

/* Temporal gauge (reading 33; not in the paper): g(x,t) = prod_{t' < t} U_t(x,t'), U'_mu(x) = g(x) U_mu(x) g(x+mu)^dag (periodic
 * wrap; the antiperiodic sign belongs to the fermions).  U_canonical: DEVICE fp64 canonical field, transformed IN PLACE; the temporal links of
 * the slices t < T-1 are written as exactly 1 (they are 1 up to rounding), slice T-1 carries the Polyakov loop.  g_out: DEVICE fp64
 * [V][3][3][re,im], the transformation (eta' = g eta, s = g^dag s').  The result may be packed with TM_RECON_18_TG / TM_RECON_12_TG. */
int tm_gauge_fix_temporal(const tm_lattice* L, double* U_canonical, double* g_out, void* stream);

/* ---- a1: spinor pack / unpack (both parities, nrhs fields) ----------------------------------------------- */
/* psi_canonical: DEVICE fp64 [nrhs][V][4][3][2]; packed: DEVICE [nrhs][parity][...] at `prec`.
 * fp16: per-site fp32 norm = max |re|,|im| over the site's 24 reals, components stored as x/norm (RN). */
int tm_spinor_pack(const tm_lattice* L, const double* psi_canonical, int prec, int nrhs, void* packed_out, void* stream);
int tm_spinor_unpack(const tm_lattice* L, const void* packed, int prec, int nrhs, double* psi_canonical, void* stream);
/* Z2 x iZ2 noise from 2-bit codes: codes DEVICE uint8 [nrhs][V][12], bit0 = re<0, bit1 = im<0;
 * value = (+-1 +- i)/sqrt(2). */
int tm_spinor_pack_z4(const tm_lattice* L, const unsigned char* codes, int prec, int nrhs, void* packed_out, void* stream);
/* The same noise from bit-packed codes: codes3 DEVICE uint8 [nrhs][V][3]; the 24 bits of a site, little endian, hold component
 * k = spin*3 + colour in bits 2k (re < 0) and 2k+1 (im < 0): 3 bytes per site instead of 12 on the host->device path. */
int tm_spinor_pack_z4_bits(const tm_lattice* L, const unsigned char* codes3, int prec, int nrhs, void* packed_out, void* stream);

/* Z2 x iZ2 noise sources made on the device ("creation of stochastic sources ... carried out on GPUs"): source r
 * of the batch is the field the synthetic-input generator (tm_inputs, counter-based splitmix64 hash) gives for seed + r *
 * seed_stride, bit-identical to its codes passed through tm_spinor_pack_z4; nothing crosses PCIe.  packed_out: DEVICE
 * [nrhs][parity][...] at `prec`. */
int tm_noise_z4(const tm_lattice* L, unsigned long long seed, unsigned long long seed_stride, int prec, int nrhs, void* packed_out,
                void* stream);

/* ---- a2+a3: hopping term with fused local epilogue ("fused CUDA kernels, such as R_oo^-1 Dslash_oe,
 *      (R_ee - kappa^2 Dslash_eo) (and their daggered analogues)") ----------------------------------------- */
/* out (parity out_parity) = epilogue(Dslash_{out_parity <- other} in).  in/out/x: DEVICE one-parity packed spinors
 * ([rhs][...] stacked, nrhs <= TM_MAX_NRHS), gauge: DEVICE packed links.  out must not alias in.
 *   PLAIN:       out = D in                    (D = Dslash, or Dslash^dag if dagger)
 *   TWIST_INV:   out = R(+-a)^-1 D in          (a = 2 kappa mu; sign - if dagger)
 *   XPAY_TWIST:  out = R(+-a) x - kappa^2 D in (x: same parity as out)
 * flops per output site counted as 1320 / 1392 / 1416. */
int tm_dslash(const tm_lattice* L, const void* gauge, int prec, int recon, void* out, const void* in, const void* x_or_null,
              int out_parity, int dagger, int kind, double kappa, double mu, int nrhs, void* stream);
/* general epilogue: out = (p0 + i p1 g5) x + (q0 + i q1 g5) (D in), pq = {p0,p1,q0,q1}; x may be NULL iff p0=p1=0. */
int tm_dslash_general(const tm_lattice* L, const void* gauge, int prec, int recon, void* out, const void* in,
                      const void* x_or_null, int out_parity, int dagger, const double pq[4], int nrhs, void* stream);

/* ---- a4: normal operator of the asymmetric even-odd system (PAPER.md:373 Eq. A2 lhs) ---------------------- */
/* out = M_pc^dag M_pc in on `parity`, M_pc = R - kappa^2 Dslash R^-1 Dslash; tmp: DEVICE, 2 one-parity spinors of nrhs. */
int tm_MdagM(const tm_lattice* L, const void* gauge, int prec, int recon, void* out, const void* in, void* tmp, int parity,
             double kappa, double mu, int nrhs, void* stream);

/* ---- a5-a7: CG ("the inverter, which is a Conjugate Gradient (CG) solver in this work, is truncated ...
 *      |r| < 10^-2 ... or a fixed number of iterations") --------------------------------------------------- */
typedef struct {
    double kappa, mu;
    double tol;            /* stop when |r_k| <= tol |b''| (iterated residual of the normal system); 0: run max_iter */
    int max_iter;
    int mode;              /* tm_cg_mode */
    double reliable_delta; /* HP_MIXED: recompute the true residual in prec_hp when |r| drops by this factor (0 -> 0.1);
                              HP_DEFECT: relative tolerance of each inner truncated solve (0 -> 1e-3) */
    int check_every;       /* LP_TRUNCATED: > 0: the host synchronises and reads the convergence flags every this many iterations;
                              0: pipelined poll -- flags follow every iteration into pinned host memory, the host stays one
                              iteration ahead of the GPU and stops one iteration after the last rhs converged */
    int skip_true_resid;   /* LP_TRUNCATED: 1 = do not recompute |b'' - A x| after the solve (saves one M^dag M);
                              info.true_resid is then -1.  The truncated mode never uses it. */
} tm_cg_params;

typedef struct {
    int iters;             /* CG iterations performed (all in prec_lp for HP_MIXED) */
    int status;            /* tm_status of this solve */
    int reliable_updates;  /* HP_MIXED only */
    double iterated_resid; /* |r_k| / |b''| */
    double true_resid;     /* |b'' - A x| / |b''| recomputed in the HP precision (LP mode: in prec_lp arithmetic) */
} tm_cg_info;

/* Solve M(kappa,mu) s = eta on the full lattice through the even-even Schur system, x0 = 0:
 *   b' = eta_e + kappa Dslash_eo R^-1 eta_o; b'' = M_pc^dag b'; CG on M_pc^dag M_pc; s_o = R^-1 (eta_o + kappa Dslash_oe s_e).
 * HP_MIXED: eta/s packed full-lattice at prec_hp; iterations in prec_lp with reliable updates in prec_hp.
 * HP_DEFECT: eta/s packed at prec_hp; defect correction (the other mixed-precision scheme of DESIGN.md reading 10): cycles of a
 *   BATCHED truncated solve of M e = r in prec_lp to relative tolerance `reliable_delta` (0 -> 1e-3), s += e and r = eta - M s
 *   in prec_hp, until |eta - M s| <= tol |eta| on the FULL lattice for every right-hand side.  All right-hand sides share every
 *   gauge load of the inner solves.  info: iters = inner iterations, reliable_updates = cycles, true_resid = |eta - M s|/|eta|.
 * LP_TRUNCATED: eta/s packed at prec_lp, everything in prec_lp storage (fp32 arithmetic, fp64 reductions), no correction;
 *   gauge_hp may be NULL.
 * info: HOST.  The call synchronises `stream` before returning.  nrhs right-hand sides share every gauge load;
 * each has its own alpha, beta and stops updating at its own convergence (info[nrhs]). */
size_t tm_cg_workspace_bytes(const tm_lattice* L, int prec_hp, int prec_lp, int mode, int nrhs);
int tm_cg_multi(const tm_lattice* L, const void* gauge_hp, int prec_hp, const void* gauge_lp, int prec_lp, int recon,
                void* s_full, const void* eta_full, const tm_cg_params* p, int nrhs, tm_cg_info* info, void* workspace,
                size_t workspace_bytes, void* stream);
/* tm_cg == tm_cg_multi with nrhs = 1 */
int tm_cg(const tm_lattice* L, const void* gauge_hp, int prec_hp, const void* gauge_lp, int prec_lp, int recon, void* s_full,
          const void* eta_full, const tm_cg_params* p, tm_cg_info* info, void* workspace, size_t workspace_bytes, void* stream);

/* ---- a8: loop contraction (PAPER.md:116 Eq. 10; :411 colour trace, Dirac indices open) --------------------- */
/* out[rhs][n][t] = sum_{x: x4=t} a(x)^dag (Gamma_n x 1) b(x), Gamma_n = g1^b0 g2^b1 g3^b2 g4^b3, n = b0+2b1+4b2+8b3.
 * a_full, b_full: DEVICE packed full-lattice spinors [nrhs][parity][...]; out: DEVICE double [nrhs][16][T][2].
 * Fixed-order two-stage reduction (bit-reproducible). */
size_t tm_loop_workspace_bytes(const tm_lattice* L, int nrhs);
int tm_loop_contract(const tm_lattice* L, const void* a_full, const void* b_full, int prec, int nrhs, double* out,
                     void* workspace, void* stream);

/* The same contraction for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): no workspace argument -- the per-block partial sums live in a file-scope device array of
 * TM_LOOP_STATIC_BYTES (8 MiB) that every GPU which loads the library holds until the process exits.  Inputs, output, arithmetic
 * and results are those of tm_loop_contract (same kernels, bit-equal).  The call performs no cudaMalloc / cudaFree and calls no
 * allocating library routine.  Limit: tm_loop_workspace_bytes(L, nrhs) <= TM_LOOP_STATIC_BYTES, i.e. nrhs * T * nb <= 32768 with
 * nb = min(32, max(1, X*Y*Z/2048)) -- 32^3 x 64 up to 16 right-hand sides per call, 64^3 x 128 up to 8; beyond it the call returns
 * TM_ERR_STATIC_LIMIT and launches nothing.  The first call on a device looks the array's device address up
 * (cudaGetSymbolAddress, once per device, with that device current): make that first call outside stream capture.
 * ALL calls of a process share the one array per device, which keeps the contents of the last call (nothing in it has to start at
 * zero: every partial is written before it is read): two calls that overlap on one GPU (different streams, or different host
 * threads) RACE on it -- keep calls on one stream, or order them with events. */
#define TM_LOOP_STATIC_BYTES 8388608
int tm_loop_contract_static(const tm_lattice* L, const void* a_full, const void* b_full, int prec, int nrhs, double* out,
                            void* stream);

/* ---- NEXT-1: estimators built from the rows above ------------------------------------------ */
/* a8': out[rhs][n][t] = scale * sum_{x: x4=t} (g5^g5_left a)^dag (Gamma_n x 1) (g5^g5_right b), scale = scale_re + i scale_im.
 * g5 = diag(1,1,-1,-1) in the public basis.  Same buffers and workspace as tm_loop_contract (which is g5 flags 0, scale 1). */
int tm_loop_contract_ex(const tm_lattice* L, const void* a_full, const void* b_full, int prec, int nrhs, int g5_left,
                        int g5_right, double scale_re, double scale_im, double* out, void* workspace, void* stream);

/* Full (unpreconditioned) operator on packed full-lattice spinors [nrhs][parity][...]:
 *   out = M(kappa, mu) in = (1 + i 2 kappa mu g5) in - kappa Dslash in   (M^dag if dagger).  mu = 0: the Wilson operator
 *   D_W = (M_u + M_d)/2 of PAPER.md:137 Eq. (14).  out_full must not alias in_full.  Two fused dslash launches. */
int tm_M(const tm_lattice* L, const void* gauge, int prec, int recon, void* out_full, const void* in_full, double kappa,
         double mu, int dagger, int nrhs, void* stream);

/* One-end trick loops from solutions s = M(kappa,+mu)^-1 eta, s_full: DEVICE [nrhs][parity][...]:
 *   TM_ONEEND_TAU3:    out[rhs][n][t] = 2 i (2 kappa mu) sum_{x: x4=t} s^dag g5 Gamma_n s             (Eq. 13; gauge may be NULL)
 *   TM_ONEEND_GENERAL: out[rhs][n][t] = 2 sum_{x: x4=t} s^dag g5 Gamma_n g5 D_W s, D_W = M(kappa,0)   (Eq. 15)
 * Noise averages (kappa-normalised M, readings 1, 25): TAU3 -> Tr_t[M_d^-1 Gamma_n] - Tr_t[M_u^-1 Gamma_n] (the sign
 * printed in Eq. 13 belongs to s = M_d^-1 eta), GENERAL -> Tr_t[M_u^-1 Gamma_n] + Tr_t[M_d^-1 Gamma_n].
 * out: DEVICE double [nrhs][16][T][2]; workspace: DEVICE, tm_oneend_workspace_bytes(). */
typedef enum { TM_ONEEND_TAU3 = 0, TM_ONEEND_GENERAL = 1 } tm_oneend_kind;
size_t tm_oneend_workspace_bytes(const tm_lattice* L, int prec, int nrhs);
int tm_oneend_loops(const tm_lattice* L, const void* gauge, int prec, int recon, const void* s_full, int kind, double kappa,
                    double mu, int nrhs, double* out, void* workspace, size_t workspace_bytes, void* stream);

/* Truncated-solver-method combination, Eq. (8), applied to loops:
 *   out[n][t] = 1/n_hp sum_{r<n_hp} (loops_hp[r] - loops_lp_same[r]) + 1/n_lp sum_{j<n_lp} loops_lp[j]
 * loops_hp / loops_lp_same: the HP and LP loops of the SAME n_hp sources; loops_lp: the n_lp further LP sources.
 * All DEVICE double [count][16][T][2]; out DEVICE double [16][T][2].  Fixed summation order. */
int tm_tsm_combine(int T, const double* loops_hp, const double* loops_lp_same, int n_hp, const double* loops_lp, int n_lp,
                   double* out, void* stream);

/* ---- NEXT-2: the paper's contraction kernels in full (App. A.2) ------------------ */
/* "A covariant-derivative kernel was also developed to allow the calculation of one-derivative insertions".
 * out = D_mu in on the full lattice, D_mu psi(x) = 1/2 [s U_mu(x) psi(x+mu) - s U_mu(x-mu)^dag psi(x-mu)] (central difference,
 * DESIGN.md reading 27; s = antiperiodic sign of a temporal hop; spin untouched).  mu = 0..3 = x,y,z,t.
 * in_full / out_full: DEVICE packed full-lattice spinors [nrhs][parity][...], must not alias.  One-derivative loops are
 * tm_loop_contract(a, D_mu b). */
int tm_covdev(const tm_lattice* L, const void* gauge, int prec, int recon, void* out_full, const void* in_full, int mu, int nrhs,
              void* stream);

/* Colour-traced contraction with the Dirac and volume indices open:
 *   out[rhs][site][al][be] = sum_c conj(a_{al c}(site)) b_{be c}(site), site = x + X (y + Y (z + Z t)).
 * out: DEVICE double [nrhs][V][4][4][2] (the layout an FFT over the volume index takes).  Products in the
 * storage arithmetic (fp32 for fp32/fp16 fields), stored as fp64. */
int tm_contract_field(const tm_lattice* L, const void* a_full, const void* b_full, int prec, int nrhs, double* out, void* stream);

/* Momentum-projected loops (PAPER.md:421 "data is sent ... for FFT ... we usually insert here a cut-off in p^2", :427 p^2 <= 9):
 *   out[rhs][n][t][k] = sum_{xvec} exp(-i p_k . xvec) a(x)^dag Gamma_n b(x),  p_k = 2 pi (m_x/X, m_y/Y, m_z/Z)
 * (forward-DFT sign, reading 28).  The contraction is fused with a separable partial DFT for the listed momenta;
 * the contraction field never goes to memory.  momenta: HOST int [n_momenta][3] = (m_x, m_y, m_z), |m_i| <= 4 (else
 * TM_ERR_ARG); copied to the device inside the call.  out: DEVICE double [nrhs][16][T][n_momenta][2].
 * workspace: DEVICE, tm_loop_momentum_workspace_bytes(L, nrhs, n_momenta, pmax) with pmax >= max |m_i|.
 * Fixed summation order, fp64 accumulation. */
size_t tm_loop_momentum_workspace_bytes(const tm_lattice* L, int nrhs, int n_momenta, int pmax);
int tm_loop_momentum(const tm_lattice* L, const void* a_full, const void* b_full, int prec, int nrhs, const int* momenta,
                     int n_momenta, double* out, void* workspace, size_t workspace_bytes, void* stream);

/* ---- NEXT-3: time dilution and hopping-parameter expansion ---------------------------------------- */
/* Time dilution / coherent sources: out = in on the time slices with keep_slice[t] != 0, zero elsewhere.
 * keep_slice: HOST uint8 [T] (T <= 512).  in_full / out_full: DEVICE packed full-lattice [nrhs][parity][...]; may alias. */
int tm_time_dilute(const tm_lattice* L, const void* in_full, int prec, int nrhs, const unsigned char* keep_slice, void* out_full,
                   void* stream);
/* Single-time-slice contraction: out[rhs][n] = sum_{x: x4 = t0} a(x)^dag Gamma_n b(x); reads slice t0 only.
 * out: DEVICE double [nrhs][16][2]; workspace as tm_loop_contract. */
int tm_loop_contract_slice(const tm_lattice* L, const void* a_full, const void* b_full, int prec, int nrhs, int t0, double* out,
                           void* workspace, void* stream);
/* HPE, Eq. (16): M_u^-1 = B - BHB + (BH)^2 B - (BH)^3 B + (BH)^4 M_u^-1, B = (1 + i 2 kappa mu g5)^-1,
 * H = 2 kappa D = -kappa Dslash (reading 2).  out = (B H)^4 s: contracted with the source it estimates the
 * stochastic fifth term (Eq. 17).  8 fused dslash launches.  tmp_full: DEVICE scratch of the size of s_full; no aliasing. */
int tm_hpe_remainder(const tm_lattice* L, const void* gauge, int prec, int recon, void* out_full, const void* s_full, void* tmp_full,
                     double kappa, double mu, int nrhs, void* stream);
/* The exact terms of Eq. (16) for an ultra-local insertion, per site: out16[n] = Tr_{spin,colour}[Gamma_n (B - BHB + (BH)^2 B
 * - (BH)^3 B)]_{xx} = 3 tr[Gamma_n (B + kappa^2 sum_mu (B(1-g_mu)B(1+g_mu)B + B(1+g_mu)B(1-g_mu)B))]; gauge independent, odd
 * powers vanish.  Multiply by X Y Z for a time slice.  out16: HOST double [16][2].  Host arithmetic only. */
int tm_hpe_local_traces(double kappa, double mu, double* out16);

/* ---- end-to-end TSM batch with HOST buffers ("the source is sent to the GPUs for inversion and
 *      contraction, and contractions are stored back in the CPUs") ----------------------------------------- */
/* codes_host: HOST (pinned recommended) uint8 [nrhs][V][12] Z2xiZ2 codes; loops_host: HOST double [nrhs][16][T][2].
 * Copies the codes H2D, packs, runs tm_cg_multi (LP_TRUNCATED), contracts eta^dag Gamma_n s, copies the loops D2H,
 * synchronises.  workspace: DEVICE, tm_tsm_workspace_bytes(). */
size_t tm_tsm_workspace_bytes(const tm_lattice* L, int prec_lp, int nrhs);
int tm_tsm_batch_host(const tm_lattice* L, const void* gauge_lp, int prec_lp, int recon, const unsigned char* codes_host,
                      const tm_cg_params* p, int nrhs, tm_cg_info* info, double* loops_host, void* workspace,
                      size_t workspace_bytes, void* stream);

/* The same with bit-packed noise codes (tm_spinor_pack_z4_bits): codes3_host HOST uint8 [nrhs][V][3], a quarter of the bytes
 * over PCIe; identical results. */
int tm_tsm_batch_host_bits(const tm_lattice* L, const void* gauge_lp, int prec_lp, int recon, const unsigned char* codes3_host,
                           const tm_cg_params* p, int nrhs, tm_cg_info* info, double* loops_host, void* workspace,
                           size_t workspace_bytes, void* stream);

/* ---- instrumentation ------------------------------------------------------------------------------------- */
/* Number of kernels this library has launched since load (all entry points). */
unsigned long long tm_launch_count(void);
/* When enabled, every dslash-family launch is bracketed by CUDA events on its stream; tm_kernel_timing_read
 * synchronises and returns the accumulated milliseconds and launch count since the last reset. */
int tm_kernel_timing_enable(int on);
int tm_kernel_timing_read(double* ms_total, long long* launches, int reset);
/* Name and template arguments (launch shape) of the kernel that dominates the batched truncated solve -- the 12-rhs fp16
 * hopping term fed from the link cache -- as a static string.  bench.py quotes DRAM traffic from an ncu capture only while
 * the capture was made with the same string (SURVEY.md 8(d) measurement). */
const char* tm_kernel_signature(void);

#ifdef __cplusplus
}
#endif
#endif
