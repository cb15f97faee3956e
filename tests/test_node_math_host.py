"""Host-side check of the product's per-node arithmetic (csrc/lbm_node.cuh compiled with g++)
against the oracle on a 1x1x1 torus, where streaming is the identity and one oracle step is one
collision.  Covers LBGK/MRT x force/no force x D2Q9/D3Q19 x fp32/fp64 and the factored MRT
transforms against the oracle's matrix.  No GPU needed."""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

from paper_1311_2404_b200 import workloads as wl

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def host(tmp_path_factory):
    so = str(tmp_path_factory.mktemp("hostnode") / "libhostnode.so")
    subprocess.check_call(["g++", "-std=c++17", "-O1", "-ffp-contract=off", "-fPIC", "-shared", "-o", so,
                           os.path.join(HERE, "host_node_check.cpp")])
    lib = C.CDLL(so)
    lib.host_mrt_transform.argtypes = [C.c_int, C.c_int, C.c_void_p, C.c_void_p]
    lib.host_update_node.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_double,
                                     C.c_void_p, C.c_void_p, C.c_void_p]
    return lib


@pytest.mark.parametrize("lattice", [wl.D2Q9, wl.D3Q19])
def test_mrt_transforms_match_oracle_matrix(host, orc, lattice):
    M, _ = orc.mrt_matrix(lattice)
    Q = M.shape[0]
    rng = np.random.default_rng(5)
    for backward, ref in ((0, M), (1, M.T)):
        for _ in range(4):
            x = rng.normal(size=Q)
            out = np.zeros(Q)
            host.host_mrt_transform(lattice, backward, x.ctypes.data, out.ctypes.data)
            np.testing.assert_allclose(out, ref @ x, rtol=0, atol=1e-12)
    # unit vectors: every entry of M exactly
    for i in range(Q):
        x = np.zeros(Q); x[i] = 1.0
        out = np.zeros(Q)
        host.host_mrt_transform(lattice, 0, x.ctypes.data, out.ctypes.data)
        assert np.array_equal(out, M[:, i])


@pytest.mark.parametrize("lattice", [wl.D2Q9, wl.D3Q19])
@pytest.mark.parametrize("mrt", [0, 1, 2, 3])  # LBGK | MRT | regularized LBGK | LBGK + Smagorinsky
@pytest.mark.parametrize("force", [0, 1, 2])  # none | Guo (eq. 17) | Exact Difference Method (eq. 18)
@pytest.mark.parametrize("f32", [0, 1])
def test_update_node_matches_oracle_collision(host, orc, lattice, mrt, force, f32):
    if mrt == 2 and force == 1:
        pytest.skip("regularized LBGK takes a force through the EDM only (reading A23)")
    rng = np.random.default_rng(100 * lattice + 10 * mrt + force)
    Q = 9 if lattice == wl.D2Q9 else 19
    tau = 0.63
    rates = np.array(wl.mrt_rates_d2q9(tau) if lattice == wl.D2Q9 else wl.mrt_rates_d3q19(tau))
    # conserved-moment rates are given non-zero here so that the force path exercises them
    rates = np.where(rates == 0.0, 0.7, rates)
    g = np.array([3e-4, -2e-4, 1e-4 if lattice == wl.D3Q19 else 0.0]) * (force != 0)
    for trial in range(5):
        v = rng.uniform(-0.05, 0.05, 3)
        f = orc.feq(lattice, 1.0 + rng.uniform(-0.05, 0.05), v[: 2 if lattice == wl.D2Q9 else 3])
        f = f * (1.0 + rng.uniform(-0.05, 0.05, Q))          # off equilibrium
        o = orc.Oracle(lattice, [wl.BGK, wl.MRT, wl.REG, wl.LES][mrt], 1, 1, 1, smagorinsky_cs=0.17, tau=tau, rates=list(rates), force=tuple(g),
                       force_scheme=1 if force == 2 else 0)
        o.set_distributions(f.reshape(Q, 1, 1, 1))
        o.step(1)
        ref = o.get_distributions().ravel()
        out = np.zeros(Q)
        host.host_update_node(lattice, f32, mrt, force, f.ctypes.data, tau, rates.ctypes.data,
                              g.ctypes.data, out.ctypes.data)
        np.testing.assert_allclose(out, ref, rtol=0, atol=2e-7 if f32 else 1e-15)
