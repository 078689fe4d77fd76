"""CPU restatement of the METHOD (cell list + list-based erfc sum + FFT-based smooth PME), fp64, OpenMP + numpy.fft.

TEST / BENCH INFRASTRUCTURE -- not the parity oracle (that is oracle/__init__.py: O(N^2), naive DFTs) and not part of the
product path.  bench.py times it as the second CPU baseline ("method_cpu"): what the same algorithm costs on the box's
host cores.  Pinned against the oracle in tests/test_oracle_pins.py.  Only tests/ and bench.py may import it.
"""
import ctypes
import math
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cpu_method.c")
_LIB = os.path.join(_HERE, "libcpumethod.so")
_lib = None


def build(force=False):
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O3", "-std=c11", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.cm_num_threads.restype = ctypes.c_int
    return _lib


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p)


class CpuMethod:
    """Neighbour list (rebuilt on demand) and PME Coulomb evaluation of one system on the host cores."""

    def __init__(self, box, rc, alpha, grid, order, r_list):
        self.box = np.ascontiguousarray(np.broadcast_to(np.asarray(box, dtype=np.float64), (3,)))
        self.rc, self.alpha, self.order, self.r_list = float(rc), float(alpha), int(order), float(r_list)
        self.K = np.ascontiguousarray(np.broadcast_to(np.asarray(grid, dtype=np.intc), (3,)))
        self.nc = np.maximum(1, np.floor(self.box / self.r_list)).astype(np.intc)
        if (self.nc < 3).any():
            raise ValueError("CpuMethod needs at least 3 cells of the list cutoff per axis")
        self.G = self._influence()

    def _knots(self):
        p = self.order          # M_p(1..p-1) by the cardinal B-spline recursion on integer arguments
        def M(n, u):
            if n == 2:
                return max(0.0, 1.0 - abs(u - 1.0))
            return (u * M(n - 1, u) + (n - u) * M(n - 1, u - 1.0)) / (n - 1)
        return np.array([M(p, k + 1.0) for k in range(p - 1)])

    def _influence(self):
        """G(m) on the half spectrum: prod_d |b_d|^2 * exp(-pi^2 mt^2/alpha^2)/(pi V mt^2), G(0) = 0."""
        K, L = self.K, self.box
        kn = self._knots()
        b2, mt = [], []
        for d in range(3):
            m = np.arange(K[d])
            den = (kn[None, :] * np.exp(2j * np.pi * m[:, None] * np.arange(len(kn))[None, :] / K[d])).sum(axis=1)
            b2.append(1.0 / np.abs(den) ** 2)
            mt.append(np.where(m <= K[d] // 2, m, m - K[d]) / L[d])
        h = K[2] // 2 + 1
        m2 = mt[0][:, None, None] ** 2 + mt[1][None, :, None] ** 2 + mt[2][None, None, :h] ** 2
        B = b2[0][:, None, None] * b2[1][None, :, None] * b2[2][None, None, :h]
        with np.errstate(divide="ignore", invalid="ignore"):
            G = B * np.exp(-np.pi ** 2 * m2 / self.alpha ** 2) / (np.pi * np.prod(L) * m2)
        G[0, 0, 0] = 0.0
        return G

    def build_list(self, pos):
        pos = np.ascontiguousarray(pos, dtype=np.float64)
        n = len(pos)
        L = lib()
        ncells = int(np.prod(self.nc))
        self.xw = np.empty((n, 3)); self.cell_of = np.empty(n, dtype=np.int32)
        self.cell_start = np.empty(ncells + 1, dtype=np.int64); self.order_ = np.empty(n, dtype=np.int32)
        L.cm_bin(ctypes.c_int64(n), _p(pos), _p(self.box), _p(self.nc), _p(self.xw), _p(self.cell_of), _p(self.cell_start),
                 _p(self.order_))
        self.wrapcount = np.floor(pos / self.box)
        self.row_ptr = np.zeros(n + 1, dtype=np.int64)
        args = (ctypes.c_int64(n), _p(self.xw), _p(self.box), _p(self.nc), ctypes.c_double(self.r_list), _p(self.cell_of),
                _p(self.cell_start), _p(self.order_), _p(self.row_ptr))
        L.cm_rows(*args, None, None)
        tot = int(self.row_ptr[-1])
        self.col = np.empty(tot, dtype=np.int32); self.shift = np.empty((tot, 3), dtype=np.int8)
        L.cm_rows(*args, _p(self.col), _p(self.shift))
        return tot // 2

    def pairs(self):
        """Unique pairs (i < j) with the shift relative to the RAW build positions, sorted: for the pin."""
        n = len(self.row_ptr) - 1
        i = np.repeat(np.arange(n, dtype=np.int32), np.diff(self.row_ptr))
        m = i < self.col
        i, j, s = i[m], self.col[m], self.shift[m].astype(np.int64)
        s = s - self.wrapcount[j].astype(np.int64) + self.wrapcount[i].astype(np.int64)
        o = np.lexsort((j, i))
        return i[o], j[o], s[o].astype(np.int8)

    def coulomb(self, pos, q, timings=None):
        """phi, F, E at the current positions (the list may be stale by less than skin/2)."""
        import time
        pos = np.ascontiguousarray(pos, dtype=np.float64); q = np.ascontiguousarray(q, dtype=np.float64)
        n = len(q)
        L = lib()
        t0 = time.perf_counter()
        x = np.ascontiguousarray(pos - self.wrapcount * self.box)          # build-time image
        phi = np.empty(n); F = np.empty((n, 3))
        L.cm_realspace(ctypes.c_int64(n), _p(x), _p(q), _p(self.box), ctypes.c_double(self.rc), ctypes.c_double(self.alpha),
                       _p(self.row_ptr), _p(self.col), _p(self.shift), _p(phi), _p(F))
        t1 = time.perf_counter()
        K = self.K
        Q = np.empty(tuple(int(k) for k in K))
        L.cm_spread(ctypes.c_int64(n), _p(pos), _p(q), _p(self.box), _p(K), ctypes.c_int(self.order), _p(Q))
        spec = np.fft.rfftn(Q)
        spec *= self.G
        Phi = np.ascontiguousarray(np.fft.irfftn(spec, s=Q.shape, axes=(0, 1, 2)) * float(np.prod(K)))      # unnormalised inverse
        pr = np.empty(n); Fr = np.empty((n, 3))
        L.cm_gather(ctypes.c_int64(n), _p(pos), _p(q), _p(self.box), _p(K), ctypes.c_int(self.order), _p(Phi), _p(pr), _p(Fr))
        t2 = time.perf_counter()
        phi = phi + pr - 2.0 * self.alpha / math.sqrt(math.pi) * q
        F = F + Fr
        if timings is not None:
            timings["t_real_s"] = t1 - t0
            timings["t_pme_s"] = t2 - t1
        return phi, F, 0.5 * float(np.dot(q, phi))
