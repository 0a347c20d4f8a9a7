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
