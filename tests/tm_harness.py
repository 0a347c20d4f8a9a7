"""Test-side plumbing around the C ABI (device buffers, pack/unpack through the library); no arithmetic of the method."""
import numpy as np
import torch

import paper_1309_2256_b200 as tm

TOL = {8: 1e-12, 4: 1e-5, 2: 5e-3}  # north_star: relative L2 per field, fp64 / fp32 / fp16 storage


def rel(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def to_dev(a):
    """complex128 / uint8 numpy array -> contiguous device tensor (complex viewed as interleaved doubles)."""
    a = np.ascontiguousarray(a)
    if a.dtype == np.complex128:
        a = a.view(np.float64)
    return torch.from_numpy(a).cuda()


class Fields:
    """A lattice, its canonical gauge field on the device and packed copies made by tm_gauge_pack."""

    def __init__(self, dims, U, ap=True):
        self.dims = tuple(dims)
        self.L = tm.tm_lattice_create(dims, ap)
        self.V = self.L.V
        self.U_dev = to_dev(U)
        self._gauge = {}

    @classmethod
    def from_slabs(cls, dims, ap=True, slab=8):
        """Large lattices: the canonical links are generated and uploaded `slab` time slices at a time (64^3x128 = 19.3 GB)."""
        import tm_inputs as ti
        X, Y, Z, T = dims
        self = cls.__new__(cls)
        self.dims = tuple(dims)
        self.L = tm.tm_lattice_create(dims, ap)
        self.V = self.L.V
        per_t = X * Y * Z * 4 * 18
        self.U_dev = torch.empty(T * per_t, dtype=torch.float64, device="cuda")
        for t0 in range(0, T, slab):
            t1 = min(T, t0 + slab)
            self.U_dev[t0 * per_t:t1 * per_t].copy_(torch.from_numpy(ti.gauge(dims, t0=t0, t1=t1).view(np.float64).reshape(-1)))
        self._gauge = {}
        return self

    def drop_canonical(self):
        self.U_dev = None
        torch.cuda.empty_cache()

    def gauge(self, prec, recon):
        key = (prec, recon)
        if key not in self._gauge:
            buf = tm.device_buffer(tm.tm_gauge_bytes(self.L, prec, recon))
            tm.tm_gauge_pack(self.L, self.U_dev, prec, recon, buf, 1e-10)
            self._gauge[key] = buf
        return self._gauge[key]

    def pb(self, prec):
        return tm.tm_spinor_bytes(self.L, prec, 0, 1)

    def pack(self, psi, prec):
        """psi: complex128 [nrhs?][T][Z][Y][X][4][3] -> packed full-lattice device buffer [nrhs][parity][...]."""
        nrhs = psi.shape[0] if psi.ndim == 7 else 1
        buf = tm.device_buffer(tm.tm_spinor_bytes(self.L, prec, 1, nrhs))
        tm.tm_spinor_pack(self.L, to_dev(psi), prec, nrhs, buf)
        return buf

    def unpack(self, buf, prec, nrhs=None):
        X, Y, Z, T = self.dims
        n = 1 if nrhs is None else nrhs
        out = torch.empty((n, T, Z, Y, X, 4, 3, 2), dtype=torch.float64, device="cuda")
        tm.tm_spinor_unpack(self.L, buf, prec, n, out)
        torch.cuda.synchronize()
        a = out.cpu().numpy().view(np.complex128)[..., 0]
        return a[0] if nrhs is None else a

    def zeros_full(self, prec, nrhs=1):
        buf = tm.device_buffer(tm.tm_spinor_bytes(self.L, prec, 1, nrhs))
        buf.zero_()
        return buf

    def half(self, full, prec, parity, nrhs=1):
        """One-parity stack [rhs][pb] (contiguous copy for nrhs > 1, a view for nrhs == 1)."""
        pb = self.pb(prec)
        if nrhs == 1:
            return full[parity * pb:(parity + 1) * pb]
        stack = tm.device_buffer(pb * nrhs)
        stack.view(nrhs, pb).copy_(full.view(nrhs, 2, pb)[:, parity, :])
        return stack

    def put_half(self, full, stack, prec, parity, nrhs):
        pb = self.pb(prec)
        full.view(nrhs, 2, pb)[:, parity, :].copy_(stack.view(nrhs, pb))


def gather_site_inputs(dims, sites, noise_seed, ap=True):
    """Geometry only: for each global site index x the inputs of the single-site hop (oracle.hop_gathered):
    U_mu(x), U_mu(x-mu), psi(x+mu), psi(x-mu) from the counter-based generators, and the temporal boundary signs.
    Returns Ufwd[N][4][3][3], Ubwd[N][4][3][3], nf[N][4][4][3], nb[N][4][4][3], sf[N][4], sb[N][4]."""
    import tm_inputs as ti
    X, Y, Z, T = dims
    sites = np.asarray(sites, dtype=np.int64)
    c = [sites % X, (sites // X) % Y, (sites // (X * Y)) % Z, sites // (X * Y * Z)]
    ext = [X, Y, Z, T]
    stride = [1, X, X * Y, X * Y * Z]
    N = sites.size
    Ufwd = ti.gauge_sites(sites)
    Ubwd = np.empty((N, 4, 3, 3), dtype=np.complex128)
    nf = np.empty((N, 4, 4, 3), dtype=np.complex128)
    nb = np.empty((N, 4, 4, 3), dtype=np.complex128)
    sf = np.ones((N, 4))
    sb = np.ones((N, 4))
    for mu in range(4):
        up = sites + np.where(c[mu] == ext[mu] - 1, -(ext[mu] - 1), 1) * stride[mu]
        dn = sites + np.where(c[mu] == 0, ext[mu] - 1, -1) * stride[mu]
        nf[:, mu] = ti.z4_sites(up, seed=noise_seed)
        nb[:, mu] = ti.z4_sites(dn, seed=noise_seed)
        Ubwd[:, mu] = ti.gauge_sites(dn)[:, mu]
    if ap:
        sf[:, 3] = np.where(c[3] == T - 1, -1.0, 1.0)
        sb[:, 3] = np.where(c[3] == 0, -1.0, 1.0)
    return Ufwd, Ubwd, nf, nb, sf, sb
