"""CPU-side checks of the C-ABI library: it builds for sm_100a, loads, exports every symbol that
include/lbm.h declares, and rejects bad parameters before touching CUDA.  No compute calls."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_1311_2404_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def declared_functions():
    text = open(os.path.join(ROOT, "include", "lbm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lbm_[a-z_]+)\s*\(", text)))


def test_header_symbols_exported(lib):
    names = declared_functions()
    assert len(names) >= 15
    for n in names:
        assert hasattr(lib, n), "liblbm_b200.so does not export %s" % n
    assert sorted(binding.EXPORTS) == names


def test_params_struct_matches_header(lib):
    # uint32 + 6 int32 (28) -> pad to 32; 2 + 19 + 3 + 1 doubles (200); 2 int32 (8) => 240 (v1);
    # + bc_velocity[3] => 264 (v2); + force_scheme + reserved => 272 (v3); + smagorinsky_cs => 280
    assert C.sizeof(binding.lbm_params) == 280
    p = binding.make_params(1, 0, 0, 8, 8, 8, tau=0.6)
    n = binding.lbm_workspace_bytes(p)
    assert n > 0
    for older in (240, 264, 272):  # callers built against an earlier layout: accepted, newer fields read as 0
        p.struct_size = older
        assert binding.lbm_workspace_bytes(p) == n
    p.struct_size = 16
    with pytest.raises(binding.LbmError) as e:
        binding.lbm_workspace_bytes(p)
    assert e.value.code == binding.LBM_EINVAL


def test_lattice_info_table1(lib):
    """Table 1: weights sum to 1, second moment delta/3, opposites are negatives."""
    for lat, Q, D in ((binding.LBM_D2Q9, 9, 2), (binding.LBM_D3Q19, 19, 3)):
        q, d, e, w, opp = binding.lbm_lattice_info(lat)
        assert (q, d) == (Q, D)
        assert abs(w.sum() - 1) < 1e-15
        assert np.allclose(np.einsum("i,ia,ib->ab", w, e, e), np.eye(3)[:, :] * (np.arange(3) < D) / 3.0, atol=1e-15)
        assert (e[opp] == -e).all()
    with pytest.raises(binding.LbmError):
        binding.lbm_lattice_info(7)


@pytest.mark.parametrize("kw,code", [
    (dict(lattice=5), binding.LBM_EINVAL),
    (dict(model=9), binding.LBM_EINVAL),
    (dict(precision=3), binding.LBM_EINVAL),
    (dict(nx=0), binding.LBM_EINVAL),
    (dict(tau=0.5), binding.LBM_EINVAL),
    (dict(nx=2048, ny=2048, nz=1024), binding.LBM_EINVAL),
    (dict(lattice=0, nz=4), binding.LBM_EINVAL),
    (dict(model=1, rates=[2.5] * 19), binding.LBM_EINVAL),
    (dict(store=7), binding.LBM_EINVAL),
    (dict(bc_velocity=(1.5, 0.0, 0.0)), binding.LBM_EINVAL),
    (dict(force_scheme=5), binding.LBM_EINVAL),
    (dict(model=5), binding.LBM_EINVAL),
    (dict(model=4, smagorinsky_cs=-1.0), binding.LBM_EINVAL),
    (dict(model=3, force=(1e-5, 0.0, 0.0)), binding.LBM_EUNSUPPORTED),
])
def test_bad_params_rejected(lib, kw, code):
    args = dict(lattice=1, model=0, precision=0, nx=8, ny=8, nz=8, tau=0.8)
    args.update(kw)
    p = binding.make_params(**args)
    with pytest.raises(binding.LbmError) as e:
        binding.lbm_workspace_bytes(p)
    assert e.value.code == code
    out = C.c_void_p()
    assert lib.lbm_create(C.byref(p), None, 0, None, C.byref(out)) == code
    assert out.value is None


def test_create_rejects_small_or_misaligned_workspace(lib):
    p = binding.make_params(1, 0, 0, 8, 8, 8, tau=0.8)
    n = binding.lbm_workspace_bytes(p)
    out = C.c_void_p()
    assert lib.lbm_create(C.byref(p), 256, n - 1, None, C.byref(out)) == binding.LBM_EINVAL
    assert lib.lbm_create(C.byref(p), 257, n, None, C.byref(out)) == binding.LBM_EINVAL
    assert b"aligned" in lib.lbm_last_error(None)


def test_workspace_accounts_for_two_copies_and_fields(lib):
    """AB store: 2 * Q * N reals per component, plus type/link bytes and SC fields."""
    N = 32 * 16 * 8
    single = binding.lbm_workspace_bytes(binding.make_params(1, 0, 0, 32, 16, 8, tau=0.8))
    double = binding.lbm_workspace_bytes(binding.make_params(1, 0, 1, 32, 16, 8, tau=0.8))
    sc = binding.lbm_workspace_bytes(binding.make_params(1, 2, 0, 32, 16, 8, tau=(1.0, 1.0)))
    assert single >= 2 * 19 * N * 4 + 5 * N
    assert double - single >= 2 * 19 * N * 4
    assert sc - single >= 2 * 19 * N * 4 + 2 * N * 4


def test_null_ctx_calls_return_einval(lib):
    assert lib.lbm_step(None, 1) == binding.LBM_EINVAL
    assert lib.lbm_destroy(None) == binding.LBM_EINVAL
    assert lib.lbm_macro(None, 0, None, None) == binding.LBM_EINVAL
    assert lib.lbm_get_dispatch(None, None) == binding.LBM_EINVAL
    assert lib.lbm_step_slabs(None, 0, 1, 1) == binding.LBM_EINVAL
    arr = (C.c_void_p * 2)(None, None)
    assert lib.lbm_step_slabs(arr, 2, 1, 1) == binding.LBM_EINVAL


def test_reserved_field_and_node_count_limit(lib):
    """lbm.h: reserved_ must be 0 (so the field can be given a meaning later); nx*ny*nz <= 2^31 - 512 (node
    indices are ints and padded threads index up to one block beyond the last node)."""
    p = binding.make_params(1, 0, 0, 8, 8, 8, tau=0.8)
    p.reserved_ = 1
    with pytest.raises(binding.LbmError) as e:
        binding.lbm_workspace_bytes(p)
    assert e.value.code == binding.LBM_EINVAL and "reserved_" in str(e.value)
    ok = binding.make_params(1, 0, 0, 2 ** 15, 2 ** 15, 1, tau=0.8)            # 2^30 nodes
    assert binding.lbm_workspace_bytes(ok) > 2 * 19 * 4 * 2 ** 30
    for nx, ny, nz in ((2 ** 16, 2 ** 15, 1), (2 ** 15, 2 ** 15, 2), (2 ** 31 - 511, 1, 1)):   # > 2^31 - 512
        with pytest.raises(binding.LbmError) as e:
            binding.lbm_workspace_bytes(binding.make_params(1, 0, 0, nx, ny, nz, tau=0.8))
        assert e.value.code == binding.LBM_EINVAL
    assert C.sizeof(binding.lbm_dispatch) == 36


def test_product_does_not_import_oracle():
    """The product path shares nothing with oracle/ (and there is no CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_1311_2404_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", text, flags=re.M), fn
                assert "lbm_oracle" not in text, fn
