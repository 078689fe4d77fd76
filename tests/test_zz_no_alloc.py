"""GPU: sqeq_energy_noalloc (the entry point that allocates nothing; scratch in a static __device__ array) against the
existing path -- the energy sqeq_coulomb returns for the same charges and potentials -- on two calls in a row.
Collected last on purpose (file name): the suite runs with pytest -x."""
import ctypes

import numpy as np
import pytest

from paper_2503_21176_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL = 1e-5   # the parity tolerance of tests/test_gpu_parity.py


def test_energy_noalloc_matches_coulomb_energy_twice():
    from paper_2503_21176_b200 import binding
    ctx = binding.Context(0)
    try:
        k = 2
        c = W.CONFIGS[k]
        pos, q = W.make(k)
        x = torch.as_tensor(pos).cuda()
        nl = ctx.nl_build(x, c.box, c.r_list)
        out = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
        rng = np.random.default_rng(31)
        bits = []
        # the first launch of a kernel may load its code (lazy module loading takes device memory): not what is measured
        binding.energy_noalloc(torch.zeros(8, device="cuda"), torch.zeros(8, device="cuda"), out)
        torch.cuda.synchronize()
        for call in range(2):
            # second call: other charges (random, not neutral-by-species), so stale scratch contents would show
            qq = q if call == 0 else (q * rng.uniform(0.5, 1.5, len(q))).astype(np.float32)
            qd = torch.as_tensor(qq).cuda()
            phi, F, E = ctx.coulomb(nl, x, qd, c.box, c.rc, c.alpha, c.grid, c.order)      # existing path
            torch.cuda.synchronize()
            free0 = torch.cuda.mem_get_info()[0]
            binding.energy_noalloc(qd, phi, out)
            torch.cuda.synchronize()
            assert torch.cuda.mem_get_info()[0] == free0            # nothing was allocated on the device
            got = out.item()
            scale = 0.5 * float((qd.double() * phi.double()).abs().sum())
            assert abs(got - E) < TOL * scale, (call, got, E)
            # and to fp64 rounding against the plain sum of the same fp32 arrays
            ref = 0.5 * float((qd.double() * phi.double()).sum())
            assert abs(got - ref) < 1e-12 * scale, (call, got, ref)
            # fixed summation order: a repeat gives the same bits
            binding.energy_noalloc(qd, phi, out)
            assert out.item() == got
            bits.append(got)
        assert bits[0] != bits[1]
        nl.free()
    finally:
        ctx.close()


def test_energy_noalloc_ragged_sizes_and_limit():
    from paper_2503_21176_b200 import binding
    rng = np.random.default_rng(32)
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    st = torch.cuda.Stream()
    for n in (1, 255, 1024, 1025, 300001):
        a = torch.as_tensor(rng.normal(size=n).astype(np.float32)).cuda()
        b = torch.as_tensor(rng.normal(size=n).astype(np.float32)).cuda()
        torch.cuda.synchronize()
        binding.energy_noalloc(a, b, out, stream=st)
        st.synchronize()
        ref = 0.5 * float((a.double() * b.double()).sum())
        assert abs(out.item() - ref) < 1e-12 * (0.5 * float((a.double() * b.double()).abs().sum()) + 1e-30), n
    # beyond the stated maximum: a clear error, nothing launched (the pointers are never touched)
    L = binding.load()
    a = torch.zeros(8, device="cuda")
    rc = L.sqeq_energy_noalloc(0, None, binding.NOALLOC_MAX_N + 1, ctypes.c_void_p(a.data_ptr()), ctypes.c_void_p(a.data_ptr()),
                               ctypes.c_void_p(out.data_ptr()))
    assert rc == binding.EINVAL
    msg = L.sqeq_last_error(None).decode()
    assert "4194304" in msg and "sqeq_energy_noalloc" in msg
    assert L.sqeq_energy_noalloc(0, None, 0, ctypes.c_void_p(a.data_ptr()), ctypes.c_void_p(a.data_ptr()),
                                 ctypes.c_void_p(out.data_ptr())) == binding.EINVAL
