"""A CPU stand-in for Context whose every tensor operation is the ORACLE's (oracle.contract / add / permsum): lets the
`-m "not gpu"` tests run the product's driver programs (ccd.py: pure call sequencing, no arithmetic) on the host and compare
the call list's result with the unfactorised equations.  Test infrastructure only."""
import numpy as np

import oracle
from oracle import sym
from gpu_util import expand_antisym_spec


class OTensor:
    def __init__(self, host):
        self.host = np.asfortranarray(np.asarray(host, dtype=np.complex128))
        self.extents = self.host.shape

    def destroy(self):
        pass


class OracleContext:
    def __init__(self):
        self.calls = 0

    def tensor_create(self, extents, zero=True):
        return OTensor(np.zeros(tuple(extents), dtype=np.complex128, order="F"))

    def tensor_from_numpy(self, x):
        return OTensor(np.array(x, dtype=np.complex128, order="F"))

    def tensor_download(self, t):
        return t.host.copy(order="F")

    def contract(self, expr, D, L, R, alpha=1.0):
        D.host = oracle.contract(expr, D.host, L.host, R.host, alpha, want_snorm=False)[0].reshape(D.host.shape)
        self.calls += 1

    def add(self, expr, D, L, alpha=1.0):
        acc = "+=" in expr
        base = D.host if acc else np.zeros_like(D.host)
        D.host = oracle.add(expr if acc else expr.replace("=", "+=", 1), base, L.host, alpha)
        self.calls += 1

    def permsum(self, D, X, perms, coefs, beta=1.0):
        D.host = oracle.permsum(D.host, X.host, perms, coefs, beta)
        self.calls += 1

    def antisymmetrize(self, spec, D, X, alpha=1.0):
        perms, signs, acc = expand_antisym_spec(spec)
        D.host = oracle.permsum(D.host, X.host, perms, [alpha * s for s in signs], 1.0 if acc else 0.0)
        self.calls += 1

    def packed_extent(self, n, k):
        return sym.packed_extent(n, k)

    def pack(self, spec, D, L):
        D.host = sym.pack(spec, L.host)
        assert D.host.shape == tuple(D.extents), (spec, D.host.shape, D.extents)
        self.calls += 1

    def unpack(self, spec, D, L, alpha=1.0):
        D.host = sym.unpack(spec, L.host, D.host, alpha)
        self.calls += 1

    def antisym_pack(self, spec, D, L, alpha=1.0):
        D.host = sym.antisym_pack(spec, L.host, D.host, alpha)
        self.calls += 1

    def denominator_divide(self, T, R, eps, alpha=1.0):
        from oracle import cc
        T.host = cc.denominator_update(np.zeros_like(R.host), R.host, eps, alpha)
        self.calls += 1

    def denominator_update(self, T, R, eps, alpha=1.0):
        from oracle import cc
        T.host = cc.denominator_update(T.host, R.host, eps, alpha)
        self.calls += 1

    def dot(self, D, X, Y, conjugate_x=True, alpha=1.0):
        x = np.conj(X.host) if conjugate_x else X.host
        D.host = np.asfortranarray(np.array(alpha * np.sum(x * Y.host)))
        self.calls += 1
