// tm_pack.cu -- a0 / a1 of SURVEY.md 8(a): canonical fp64 fields <-> packed even-odd SoA at fp64/fp32/fp16.
#include <mutex>
#include "tm_layout.cuh"

namespace tmk {

__device__ unsigned int g_su3_dev_bits; // max deviation from SU(3) seen by the last gauge pack (float bits)
__device__ unsigned int g_r8_inv_bits;  // recon 8: max 1 / (|U01|^2 + |U02|^2) seen by the last gauge pack (float bits)
__device__ unsigned int g_tg_bad;       // *_TG codes: number of temporal links of slices t < T-1 that are not exactly the unit matrix

template <int PREC, bool FX = false> // FX: 16-bit fixed-point words (TM_RECON_*_FIX16, tm.h) instead of binary16
__device__ __forceinline__ void store_reals(void* block, int Vh, int cb, const double* u, int n)
{
    // generic element-wise store following the chunk layout of tm_layout.cuh (n reals per site)
    const int w = PREC;
    const int bytes = n * w;
    const int nfull = bytes / 16;      // 16-byte chunks
    const int per = 16 / w;            // reals per full chunk
    char* base = static_cast<char*>(block);
    for (int r = 0; r < n; ++r) {
        char* dst;
        if (r < nfull * per) {
            dst = base + ((size_t)(r / per) * Vh + cb) * 16 + (size_t)(r % per) * w;
        } else {
            const int tail_reals = n - nfull * per; // reals in the tail array
            dst = base + (size_t)nfull * Vh * 16 + ((size_t)cb * tail_reals + (r - nfull * per)) * w;
        }
        if (PREC == 8) *reinterpret_cast<double*>(dst) = u[r];
        else if (PREC == 4) *reinterpret_cast<float*>(dst) = (float)u[r];
        else if (FX) *reinterpret_cast<unsigned short*>(dst) = (unsigned short)(32768 + (int)rint(fmin(1.0, fmax(-1.0, u[r])) * 32767.0));
        else *reinterpret_cast<__half*>(dst) = __float2half_rn((float)u[r]);
    }
}

template <int PREC, int RECON_CODE>
__global__ void gauge_pack_kernel(Geo g, const double* __restrict__ U, char* out, size_t link_block, int check, int tgcheck)
{
    constexpr int RECON = RECON_CODE % 100;
    constexpr bool FX = RECON_CODE >= 100 && PREC == 2;
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    const int pm = blockIdx.y; // parity*4 + mu
    if (cb >= g.Vh) return;
    const int parity = pm >> 2, mu = pm & 3;
    uint32_t row, xh, rem2, y, t, z;
    g.dXh.divmod((uint32_t)cb, row, xh);
    g.dY.divmod(row, rem2, y);
    g.dZ.divmod(rem2, t, z);
    const int xodd = (parity + y + z + t) & 1;
    const size_t site = 2 * (size_t)cb + xodd;
    double u[18];
#pragma unroll
    for (int k = 0; k < 18; ++k) u[k] = U[(site * 4 + mu) * 18 + k];
    if (tgcheck && mu == 3 && (int)t < g.T - 1) { // declared temporal gauge (tm.h): exactly the unit matrix
        bool one = true;
        for (int k = 0; k < 18; ++k) one = one && (u[k] == ((k == 0 || k == 8 || k == 16) ? 1.0 : 0.0));
        if (!one) atomicAdd(&g_tg_bad, 1u);
    }
    if (check) {
        // deviation from SU(3): |U U^dag - 1|_max and |row2 - conj(row0 x row1)|_max
        double dev = 0;
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) {
                double re = 0, im = 0;
                for (int c = 0; c < 3; ++c) {
                    const double ar = u[2 * (a * 3 + c)], ai = u[2 * (a * 3 + c) + 1];
                    const double br = u[2 * (b * 3 + c)], bi = u[2 * (b * 3 + c) + 1];
                    re += ar * br + ai * bi;
                    im += ai * br - ar * bi;
                }
                dev = fmax(dev, fmax(fabs(re - (a == b ? 1.0 : 0.0)), fabs(im)));
            }
        double w[18];
        for (int k = 0; k < 12; ++k) w[k] = u[k];
        rebuild_row2(w);
        for (int k = 12; k < 18; ++k) dev = fmax(dev, fabs(w[k] - u[k]));
        if (!(dev == dev)) dev = 1e30; // NaN
        atomicMax(&g_su3_dev_bits, __float_as_uint((float)dev));
    }
    if (RECON == 8) { // V01, V02, V10, arg(V00)/pi, arg(V20)/pi of V_ij = U_{i,(j+2)%3} (tm_layout.cuh rebuild_from8)
        double v[18];
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j) {
                v[2 * (i * 3 + j)] = u[2 * (i * 3 + (j + 2) % 3)];
                v[2 * (i * 3 + j) + 1] = u[2 * (i * 3 + (j + 2) % 3) + 1];
            }
        const double r8 = v[2] * v[2] + v[3] * v[3] + v[4] * v[4] + v[5] * v[5];
        atomicMax(&g_r8_inv_bits, __float_as_uint(r8 > 1e-30 ? (float)fmin(1.0 / r8, 1e30) : 1e30f));
        double q[8] = {v[2], v[3], v[4], v[5], v[6], v[7], atan2(v[1], v[0]) / 3.14159265358979323846, atan2(v[13], v[12]) / 3.14159265358979323846};
        store_reals<PREC>(out + (size_t)pm * link_block, g.Vh, cb, q, 8);
        return;
    }
    store_reals<PREC, FX>(out + (size_t)pm * link_block, g.Vh, cb, u, RECON);
}

template <int PREC, int MODE> // MODE 0: pack from fp64 canonical, 1: unpack to fp64 canonical, 2: pack from Z2xiZ2 codes (one byte
                              // per component), 3: from bit-packed codes (3 bytes per site: component k in bits 2k, 2k+1)
__global__ void spinor_pack_kernel(Geo g, const double* __restrict__ src, double* dst, const unsigned char* __restrict__ codes,
                                   char* packed, size_t parity_bytes, long long V)
{
    typedef typename Prec<PREC>::real real;
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    const int parity = blockIdx.y, rhs = blockIdx.z;
    if (cb >= g.Vh) return;
    uint32_t row, xh, rem2, y, t, z;
    g.dXh.divmod((uint32_t)cb, row, xh);
    g.dY.divmod(row, rem2, y);
    g.dZ.divmod(rem2, t, z);
    const int xodd = (parity + y + z + t) & 1;
    const size_t site = (size_t)rhs * V + 2 * (size_t)cb + xodd;
    char* field = packed + ((size_t)rhs * 2 + parity) * parity_bytes;
    real v[24];
    if (MODE == 0) {
#pragma unroll
        for (int k = 0; k < 24; ++k) v[k] = (real)src[site * 24 + k];
        store_spinor<PREC>(field, g.Vh, cb, v);
    } else if (MODE == 2) {
        const real r = (real)0.70710678118654752440;
#pragma unroll
        for (int k = 0; k < 12; ++k) {
            const unsigned c = codes[site * 12 + k];
            v[2 * k] = (c & 1u) ? -r : r;
            v[2 * k + 1] = (c & 2u) ? -r : r;
        }
        store_spinor<PREC>(field, g.Vh, cb, v);
    } else if (MODE == 3) {
        const real r = (real)0.70710678118654752440;
        const unsigned w = (unsigned)codes[site * 3] | ((unsigned)codes[site * 3 + 1] << 8) | ((unsigned)codes[site * 3 + 2] << 16);
#pragma unroll
        for (int k = 0; k < 12; ++k) {
            v[2 * k] = ((w >> (2 * k)) & 1u) ? -r : r;
            v[2 * k + 1] = ((w >> (2 * k + 1)) & 1u) ? -r : r;
        }
        store_spinor<PREC>(field, g.Vh, cb, v);
    } else {
        load_spinor<PREC>(field, g.Vh, cb, v);
#pragma unroll
        for (int k = 0; k < 24; ++k) dst[site * 24 + k] = (double)v[k];
    }
}

// ---- Z2 x iZ2 noise made on the device ("creation of stochastic sources ... carried out on GPUs") ------------
// The library's own statement of the counter-based generator of the synthetic inputs (three chained splitmix64 rounds over
// (seed, stream 2, site * 12 + component, draw 0); the two top bits are the signs of re and im): source r of a batch is the
// field of seed + r * seed_stride, bit-identical to the host generator's codes fed through tm_spinor_pack_z4.
__device__ __forceinline__ unsigned long long dev_splitmix64(unsigned long long z)
{
    z += 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

template <int PREC>
__global__ void noise_z4_kernel(Geo g, unsigned long long seed, unsigned long long seed_stride, char* packed, size_t parity_bytes)
{
    typedef typename Prec<PREC>::real real;
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    const int parity = blockIdx.y, rhs = blockIdx.z;
    if (cb >= g.Vh) return;
    uint32_t row, xh, rem2, y, t, z;
    g.dXh.divmod((uint32_t)cb, row, xh);
    g.dY.divmod(row, rem2, y);
    g.dZ.divmod(rem2, t, z);
    const unsigned long long site = 2ull * (unsigned long long)cb + ((parity + y + z + t) & 1);
    const unsigned long long s0 = dev_splitmix64((seed + (unsigned long long)rhs * seed_stride) ^ (2ull * 0xD6E8FEB86659FD93ULL));
    const real r = (real)0.70710678118654752440;
    real v[24];
#pragma unroll
    for (int k = 0; k < 12; ++k) {
        unsigned long long h = dev_splitmix64(s0 ^ ((site * 12ull + (unsigned long long)k) * 0xA0761D6478BD642FULL));
        h = dev_splitmix64(h); // draw 0: h ^ (0 * constant)
        const unsigned code = (unsigned)(h >> 62);
        v[2 * k] = (code & 1u) ? -r : r;
        v[2 * k + 1] = (code & 2u) ? -r : r;
    }
    store_spinor<PREC>(packed + ((size_t)rhs * 2 + parity) * parity_bytes, g.Vh, cb, v);
}

// ---- synthetic SU(3) gauge field made on the device (SURVEY.md 8(f) NEXT-4 "on-device noise/gauge generators") --------------
// The library's own statement of the link generator of the synthetic inputs: hashes (seed, stream 1,
// link = 4 site + mu, draw 0..17) -> nine Box-Muller pairs -> A = w 1 + eps G -> Gram-Schmidt rows 0, 1 -> row 2 = conj(row0 x row1).
// The hashes are bit-identical to the host generator's; log / cos / sin / sqrt are the device's fp64 routines and the products
// may be contracted into FMAs, so the links agree with the host's to rounding (tm.h states the tolerance), not bit for bit.
__device__ __forceinline__ double dev_u01(unsigned long long h) { return ((double)(h >> 11) + 1.0) * (1.0 / 9007199254740992.0); }

__global__ void __launch_bounds__(128) gauge_synth_kernel(long long nlinks, unsigned long long seed, double w, double eps, double* __restrict__ U)
{
    const long long link = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (link >= nlinks) return;
    const unsigned long long s0 = dev_splitmix64(seed ^ (1ull * 0xD6E8FEB86659FD93ULL));
    const unsigned long long s1 = dev_splitmix64(s0 ^ ((unsigned long long)link * 0xA0761D6478BD642FULL));
    double a[3][3][2];
    for (int k = 0; k < 9; ++k) {
        const unsigned long long h1 = dev_splitmix64(s1 ^ ((unsigned long long)(2 * k) * 0xE7037ED1A0B428DBULL));
        const unsigned long long h2 = dev_splitmix64(s1 ^ ((unsigned long long)(2 * k + 1) * 0xE7037ED1A0B428DBULL));
        const double r = sqrt(-2.0 * log(dev_u01(h1)));
        const double ph = 6.283185307179586476925286766559 * dev_u01(h2);
        double sn, cs;
        sincos(ph, &sn, &cs);
        a[k / 3][k % 3][0] = eps * (r * cs) + ((k / 3 == k % 3) ? w : 0.0);
        a[k / 3][k % 3][1] = eps * (r * sn);
    }
    double n = 0;
    for (int j = 0; j < 3; ++j) n += a[0][j][0] * a[0][j][0] + a[0][j][1] * a[0][j][1];
    n = 1.0 / sqrt(n);
    for (int j = 0; j < 3; ++j) { a[0][j][0] *= n; a[0][j][1] *= n; }
    double pr = 0, pi = 0; // row0^dagger . row1
    for (int j = 0; j < 3; ++j) {
        pr += a[0][j][0] * a[1][j][0] + a[0][j][1] * a[1][j][1];
        pi += a[0][j][0] * a[1][j][1] - a[0][j][1] * a[1][j][0];
    }
    for (int j = 0; j < 3; ++j) {
        a[1][j][0] -= pr * a[0][j][0] - pi * a[0][j][1];
        a[1][j][1] -= pr * a[0][j][1] + pi * a[0][j][0];
    }
    n = 0;
    for (int j = 0; j < 3; ++j) n += a[1][j][0] * a[1][j][0] + a[1][j][1] * a[1][j][1];
    n = 1.0 / sqrt(n);
    for (int j = 0; j < 3; ++j) { a[1][j][0] *= n; a[1][j][1] *= n; }
    for (int j = 0; j < 3; ++j) {
        const int j1 = (j + 1) % 3, j2 = (j + 2) % 3;
        a[2][j][0] = (a[0][j1][0] * a[1][j2][0] - a[0][j1][1] * a[1][j2][1]) - (a[0][j2][0] * a[1][j1][0] - a[0][j2][1] * a[1][j1][1]);
        a[2][j][1] = -((a[0][j1][0] * a[1][j2][1] + a[0][j1][1] * a[1][j2][0]) - (a[0][j2][0] * a[1][j1][1] + a[0][j2][1] * a[1][j1][0]));
    }
    double2* dst = reinterpret_cast<double2*>(U + link * 18);
    for (int k = 0; k < 9; ++k) dst[k] = make_double2(a[k / 3][k % 3][0], a[k / 3][k % 3][1]);
}

// ---- temporal gauge (tm.h: tm_gauge_fix_temporal) -------------------------------------------------------------------------
__device__ __forceinline__ void cmat_mul(const double* a, const double* b, double* c, bool bdag) // c = a b  or  a b^dag
{
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            double re = 0.0, im = 0.0;
            for (int k = 0; k < 3; ++k) {
                const double ar = a[2 * (i * 3 + k)], ai = a[2 * (i * 3 + k) + 1];
                const double br = bdag ? b[2 * (j * 3 + k)] : b[2 * (k * 3 + j)];
                const double bi = bdag ? -b[2 * (j * 3 + k) + 1] : b[2 * (k * 3 + j) + 1];
                re += ar * br - ai * bi;
                im += ar * bi + ai * br;
            }
            c[2 * (i * 3 + j)] = re;
            c[2 * (i * 3 + j) + 1] = im;
        }
}

// one thread per spatial site: g(x, 0) = 1, g(x, t + 1) = g(x, t) U_t(x, t)
__global__ void tgauge_g_kernel(Geo g, const double* __restrict__ U, double* __restrict__ G)
{
    const long long v3 = (long long)g.X * g.Y * g.Z;
    const long long xs = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (xs >= v3) return;
    double cur[18], nxt[18];
    for (int k = 0; k < 18; ++k) cur[k] = (k == 0 || k == 8 || k == 16) ? 1.0 : 0.0;
    for (int t = 0; t < g.T; ++t) {
        const long long site = xs + v3 * t;
        for (int k = 0; k < 18; ++k) G[site * 18 + k] = cur[k];
        cmat_mul(cur, U + (site * 4 + 3) * 18, nxt, false);
        for (int k = 0; k < 18; ++k) cur[k] = nxt[k];
    }
}

// one thread per (site, mu): U'_mu(x) = g(x) U_mu(x) g(x + mu)^dag in place; temporal links inside the lattice are set to exactly 1
__global__ void tgauge_apply_kernel(Geo g, double* U, const double* __restrict__ G, long long V)
{
    const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= 4 * V) return;
    const long long site = id >> 2;
    const int mu = (int)(id & 3);
    const int ext[4] = {g.X, g.Y, g.Z, g.T};
    const long long stride[4] = {1, g.X, (long long)g.X * g.Y, (long long)g.X * g.Y * g.Z};
    const int c = (int)((site / stride[mu]) % ext[mu]);
    const long long up = site + (c == ext[mu] - 1 ? -(long long)(ext[mu] - 1) : 1) * stride[mu];
    double* u = U + id * 18;
    if (mu == 3 && c < g.T - 1) {
        for (int k = 0; k < 18; ++k) u[k] = (k == 0 || k == 8 || k == 16) ? 1.0 : 0.0;
        return;
    }
    double a[18], b[18];
    cmat_mul(G + site * 18, u, a, false);
    cmat_mul(a, G + up * 18, b, true);
    for (int k = 0; k < 18; ++k) u[k] = b[k];
}

template <int PREC>
static int gauge_pack_t(const Geo& g, const double* U, int recon, void* out, int check, int tgcheck, cudaStream_t st)
{
    dim3 block(128), grid((g.Vh + 127) / 128, 8);
    if (recon == 18) gauge_pack_kernel<PREC, 18><<<grid, block, 0, st>>>(g, U, (char*)out, link_block_bytes(g, PREC, 18), check, tgcheck);
    else if (recon == 8) gauge_pack_kernel<PREC, 8><<<grid, block, 0, st>>>(g, U, (char*)out, link_block_bytes(g, PREC, 8), check, tgcheck);
    else if (recon == 118) gauge_pack_kernel<PREC, 118><<<grid, block, 0, st>>>(g, U, (char*)out, link_block_bytes(g, PREC, 18), check, tgcheck);
    else if (recon == 112) gauge_pack_kernel<PREC, 112><<<grid, block, 0, st>>>(g, U, (char*)out, link_block_bytes(g, PREC, 12), check, tgcheck);
    else gauge_pack_kernel<PREC, 12><<<grid, block, 0, st>>>(g, U, (char*)out, link_block_bytes(g, PREC, 12), check, tgcheck);
    TM_LAUNCH_CHECK("gauge_pack_kernel");
    return TM_OK;
}

template <int PREC>
static int spinor_pack_t(const Geo& g, long long V, int mode, const double* src, double* dst, const unsigned char* codes,
                         void* packed, int nrhs, cudaStream_t st)
{
    dim3 block(128), grid((g.Vh + 127) / 128, 2, nrhs);
    const size_t pb = spinor_parity_bytes(g, PREC);
    if (mode == 0) spinor_pack_kernel<PREC, 0><<<grid, block, 0, st>>>(g, src, dst, codes, (char*)packed, pb, V);
    else if (mode == 1) spinor_pack_kernel<PREC, 1><<<grid, block, 0, st>>>(g, src, dst, codes, (char*)packed, pb, V);
    else if (mode == 2) spinor_pack_kernel<PREC, 2><<<grid, block, 0, st>>>(g, src, dst, codes, (char*)packed, pb, V);
    else spinor_pack_kernel<PREC, 3><<<grid, block, 0, st>>>(g, src, dst, codes, (char*)packed, pb, V);
    TM_LAUNCH_CHECK("spinor_pack_kernel");
    return TM_OK;
}

int spinor_pack_any(const Geo& g, long long V, int prec, int mode, const double* src, double* dst, const unsigned char* codes,
                    void* packed, int nrhs, cudaStream_t st)
{
    if (prec == 8) return spinor_pack_t<8>(g, V, mode, src, dst, codes, packed, nrhs, st);
    if (prec == 4) return spinor_pack_t<4>(g, V, mode, src, dst, codes, packed, nrhs, st);
    return spinor_pack_t<2>(g, V, mode, src, dst, codes, packed, nrhs, st);
}

} // namespace tmk

using namespace tmk;

extern "C" int tm_gauge_fix_temporal(const tm_lattice* L, double* U, double* g_out, void* stream)
{
    if (!L || !U || !g_out) return TM_ERR_ARG;
    if (!aligned256(U) || !aligned256(g_out)) return TM_ERR_LAYOUT;
    cudaStream_t st = (cudaStream_t)stream;
    const long long v3 = (long long)L->g.X * L->g.Y * L->g.Z;
    tgauge_g_kernel<<<(unsigned)((v3 + 127) / 128), 128, 0, st>>>(L->g, U, g_out);
    TM_LAUNCH_CHECK("tgauge_g_kernel");
    tgauge_apply_kernel<<<(unsigned)((4 * L->V + 127) / 128), 128, 0, st>>>(L->g, U, g_out, L->V);
    TM_LAUNCH_CHECK("tgauge_apply_kernel");
    return TM_OK;
}

extern "C" int tm_gauge_pack(const tm_lattice* L, const double* U, int prec, int recon, void* out, double su3_tol, void* stream)
{
    if (!L || !U || !out || !valid_prec(prec) || !valid_recon(recon)) return TM_ERR_ARG;
    if (!aligned256(U) || !aligned256(out)) return TM_ERR_LAYOUT;
    cudaStream_t st = (cudaStream_t)stream;
    // the check counters are device symbols shared by every call: concurrent packs (other host threads, other streams) take turns;
    // every check below ends with a stream synchronisation inside the lock, so a counter is read before the next pack resets it
    static std::mutex pack_mu;
    std::lock_guard<std::mutex> pack_lock(pack_mu);
    const int tgcheck = recon >= 200 ? 1 : 0; // declaration only: the field is stored like the plain 18 / 12-real one
    recon = stored_recon(prec, recon);
    const int check = (recon % 100 != 18 && su3_tol > 0) ? 1 : 0;
    if (tgcheck) {
        const unsigned int zero = 0;
        TM_CUDA_CHECK(cudaMemcpyToSymbolAsync(g_tg_bad, &zero, sizeof(zero), 0, cudaMemcpyHostToDevice, st));
    }
    if (check) {
        const unsigned int zero = 0;
        TM_CUDA_CHECK(cudaMemcpyToSymbolAsync(g_su3_dev_bits, &zero, sizeof(zero), 0, cudaMemcpyHostToDevice, st));
    }
    if (recon == 8) {
        const unsigned int zero = 0;
        TM_CUDA_CHECK(cudaMemcpyToSymbolAsync(g_r8_inv_bits, &zero, sizeof(zero), 0, cudaMemcpyHostToDevice, st));
    }
    int rc;
    if (prec == 8) rc = gauge_pack_t<8>(L->g, U, recon, out, check, tgcheck, st);
    else if (prec == 4) rc = gauge_pack_t<4>(L->g, U, recon, out, check, tgcheck, st);
    else rc = gauge_pack_t<2>(L->g, U, recon, out, check, tgcheck, st);
    if (rc != TM_OK) return rc;
    if (tgcheck) { // this check always synchronises the stream
        unsigned int bad = 0;
        TM_CUDA_CHECK(cudaMemcpyFromSymbolAsync(&bad, g_tg_bad, sizeof(bad), 0, cudaMemcpyDeviceToHost, st));
        TM_CUDA_CHECK(cudaStreamSynchronize(st));
        if (bad != 0) return TM_ERR_NOT_TGAUGE;
    }
    if (check) {
        unsigned int bits = 0;
        TM_CUDA_CHECK(cudaMemcpyFromSymbolAsync(&bits, g_su3_dev_bits, sizeof(bits), 0, cudaMemcpyDeviceToHost, st));
        TM_CUDA_CHECK(cudaStreamSynchronize(st));
        float dev;
        memcpy(&dev, &bits, sizeof(dev));
        if (dev > su3_tol) return TM_ERR_NOT_SU3;
    }
    if (recon == 8) { // the 8-real chart is singular where U01 = U02 = 0 (e.g. the unit link): refuse such fields
        unsigned int bits = 0;
        TM_CUDA_CHECK(cudaMemcpyFromSymbolAsync(&bits, g_r8_inv_bits, sizeof(bits), 0, cudaMemcpyDeviceToHost, st));
        TM_CUDA_CHECK(cudaStreamSynchronize(st));
        float rinv;
        memcpy(&rinv, &bits, sizeof(rinv));
        if (rinv > 1e6f) return TM_ERR_RECON8;
    }
    return TM_OK;
}

extern "C" int tm_spinor_pack(const tm_lattice* L, const double* psi, int prec, int nrhs, void* out, void* stream)
{
    if (!L || !psi || !out || !valid_prec(prec) || nrhs < 1) return TM_ERR_ARG;
    if (!aligned256(psi) || !aligned256(out)) return TM_ERR_LAYOUT;
    return spinor_pack_any(L->g, L->V, prec, 0, psi, nullptr, nullptr, out, nrhs, (cudaStream_t)stream);
}

extern "C" int tm_spinor_unpack(const tm_lattice* L, const void* packed, int prec, int nrhs, double* psi, void* stream)
{
    if (!L || !psi || !packed || !valid_prec(prec) || nrhs < 1) return TM_ERR_ARG;
    if (!aligned256(psi) || !aligned256(packed)) return TM_ERR_LAYOUT;
    return spinor_pack_any(L->g, L->V, prec, 1, nullptr, psi, nullptr, const_cast<void*>(packed), nrhs, (cudaStream_t)stream);
}

extern "C" int tm_spinor_pack_z4(const tm_lattice* L, const unsigned char* codes, int prec, int nrhs, void* out, void* stream)
{
    if (!L || !codes || !out || !valid_prec(prec) || nrhs < 1) return TM_ERR_ARG;
    if (!aligned256(codes) || !aligned256(out)) return TM_ERR_LAYOUT;
    return spinor_pack_any(L->g, L->V, prec, 2, nullptr, nullptr, codes, out, nrhs, (cudaStream_t)stream);
}

extern "C" int tm_spinor_pack_z4_bits(const tm_lattice* L, const unsigned char* codes3, int prec, int nrhs, void* out, void* stream)
{
    if (!L || !codes3 || !out || !valid_prec(prec) || nrhs < 1) return TM_ERR_ARG;
    if (!aligned256(codes3) || !aligned256(out)) return TM_ERR_LAYOUT;
    return spinor_pack_any(L->g, L->V, prec, 3, nullptr, nullptr, codes3, out, nrhs, (cudaStream_t)stream);
}

extern "C" int tm_gauge_synthetic(const tm_lattice* L, unsigned long long seed, double w, double eps, double* U_canonical_out, void* stream)
{
    if (!L || !U_canonical_out) return TM_ERR_ARG;
    if (!aligned256(U_canonical_out)) return TM_ERR_LAYOUT;
    const long long nlinks = L->V * 4;
    gauge_synth_kernel<<<(unsigned)((nlinks + 127) / 128), 128, 0, (cudaStream_t)stream>>>(nlinks, seed, w, eps, U_canonical_out);
    TM_LAUNCH_CHECK("gauge_synth_kernel");
    return TM_OK;
}

extern "C" int tm_noise_z4(const tm_lattice* L, unsigned long long seed, unsigned long long seed_stride, int prec, int nrhs,
                           void* packed_out, void* stream)
{
    if (!L || !packed_out || !valid_prec(prec) || nrhs < 1) return TM_ERR_ARG;
    if (!aligned256(packed_out)) return TM_ERR_LAYOUT;
    const Geo& g = L->g;
    dim3 block(128), grid((g.Vh + 127) / 128, 2, nrhs);
    const size_t pb = spinor_parity_bytes(g, prec);
    cudaStream_t st = (cudaStream_t)stream;
    if (prec == 8) noise_z4_kernel<8><<<grid, block, 0, st>>>(g, seed, seed_stride, (char*)packed_out, pb);
    else if (prec == 4) noise_z4_kernel<4><<<grid, block, 0, st>>>(g, seed, seed_stride, (char*)packed_out, pb);
    else noise_z4_kernel<2><<<grid, block, 0, st>>>(g, seed, seed_stride, (char*)packed_out, pb);
    TM_LAUNCH_CHECK("noise_z4_kernel");
    return TM_OK;
}
