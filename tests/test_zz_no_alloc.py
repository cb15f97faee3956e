"""lbm_step_noalloc (include/lbm.h): the path in one call that allocates nothing -- the context's workspace is
a file-scope device array inside the library.  Its output must equal what the ordinary calls
(lbm_create on a caller-owned workspace, set_geometry, set_distributions, step, get_distributions) give for
the same inputs, within the tolerance of the parity tests (1e-5 fp32 / 1e-12 fp64; the kernels are the same,
so in fact to the bit), on calls in a row that reuse the array with other lattices in between, and the call
must not allocate device memory.  Named test_zz_* so that pytest collects it last."""
import numpy as np
import pytest

from paper_1311_2404_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = {W.F32: 1e-5, W.F64: 1e-12}


def existing_path(B, w, f_in, n):
    """Reference: the ordinary API with a torch-owned workspace."""
    import torch
    sim = B.from_workload(w)
    sim.set_geometry(w.mask)
    for s in range(w.ncomp):
        sim.set_distributions(f_in[s], comp=s)
    sim.step(n)
    out = torch.stack([sim.get_distributions(s) for s in range(w.ncomp)])
    sim.close()
    return out


def start_state(B, w, seed):
    """Canonical f[ncomp][Q][z][y][x] on the device: equilibrium of the workload's fields, knocked off equilibrium."""
    import torch
    sim = B.from_workload(w)
    sim.set_geometry(w.mask)
    for s in range(w.ncomp):
        sim.init_equilibrium(w.rho[s], w.u[s], comp=s)
    f = torch.stack([sim.get_distributions(s) for s in range(w.ncomp)])
    sim.close()
    g = torch.Generator(device="cpu").manual_seed(seed)
    bump = 1 + 0.01 * (2 * torch.rand(f.shape, generator=g, dtype=torch.float64) - 1)
    return (f * bump.to(f.device, f.dtype)).contiguous()


def noalloc(B, w, f_in, n):
    import torch
    probe = B.from_workload(w)  # the parameters exactly as the existing path builds them
    p = probe.params
    probe.close()
    mask = torch.as_tensor(w.mask).to("cuda:0").contiguous()
    out = torch.empty_like(f_in)
    B.lbm_step_noalloc(p, mask.data_ptr(), f_in.data_ptr(), out.data_ptr(), n, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return out


def generic(lattice, model, precision, shape, seed, **kw):
    nx, ny, nz = shape
    ncomp = 2 if model == W.SC2 else 1
    mask, rho, u = W.random_types(lattice, nx, ny, nz, seed, ncomp=ncomp)
    w = W.Workload("noalloc", lattice, model, precision, nx, ny, nz, kw.pop("tau", (0.7, 0.9)), 0, **kw)
    w.mask, w.rho, w.u = mask, rho, u
    return w


def cases():
    yield W.c3_mrt_obstacles(40, 24, 12, precision=W.F64), 23           # MRT, random solids, fp64
    yield W.c2_channel(64, 32, 16), 40                                  # LBGK + Guo force, fp32, V = 2 packs
    yield W.c5_shan_chen(32, 24, 16), 17                                # two components: psi / u' scratch fields too
    yield generic(W.D2Q9, W.LES, W.F32, (50, 37, 1), 5, smagorinsky_cs=0.15, force=(1e-5, -2e-5, 0.0),
                  bc_velocity=(0.02, -0.01, 0.0)), 30                   # all node types, ragged extents
    yield W.c3_mrt_obstacles(40, 24, 12, precision=W.F64), 23           # the first lattice again, over the others' leftovers


def test_noalloc_entry_matches_existing_path_on_calls_in_a_row():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1311_2404_b200 import binding as B
    B.load()
    # the static array comes with the library's module, which CUDA loads lazily at the first call: warm up once
    tiny = B.make_params(B.LBM_D3Q19, B.LBM_BGK, B.LBM_F32, 4, 4, 4, tau=0.8)
    t = torch.full((19, 4, 4, 4), 1.0 / 19, device="cuda:0")
    B.lbm_step_noalloc(tiny, None, t.data_ptr(), t.data_ptr(), 2, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert abs(float(t.sum()) - 64.0) < 1e-4                            # in place (d_f_out == d_f_in), mass kept
    first = None
    for k, (w, n) in enumerate(cases()):
        f_in = start_state(B, w, seed=100 + k % 4)                      # case 4 repeats case 0, inputs included
        want = existing_path(B, w, f_in, n)
        torch.cuda.synchronize()
        before = torch.cuda.mem_get_info()[0]
        got = noalloc(B, w, f_in, n)
        got2 = noalloc(B, w, f_in, n)                                   # two calls in a row on the same inputs
        after = torch.cuda.mem_get_info()[0]
        live = torch.as_tensor(w.mask != W.SOLID).to(got.device)
        err = (got.double() - want.double()).abs()[:, :, live].max().item()
        assert err <= TOL[w.precision], (k, w.name, err)
        assert torch.equal(got[:, :, live], want[:, :, live]), (k, w.name)     # same kernels: same bits
        assert torch.equal(got, got2), (k, w.name)
        assert (got[:, :, ~live] == 0).all()                            # SOLID nodes read back as 0, as in the existing path
        # out tensors of the two calls (torch's caching allocator) aside, the calls took no device memory
        assert before - after <= 2 * got.numel() * got.element_size() + (8 << 20), (before, after)
        if k == 0:
            first = got.clone()
    assert torch.equal(first, got)                                      # the repeat of case 0 after three other lattices


def test_noalloc_entry_rejects_what_does_not_fit_and_bad_arguments():
    import torch
    assert torch.cuda.is_available()
    from paper_1311_2404_b200 import binding as B
    B.load()
    big = B.make_params(B.LBM_D3Q19, B.LBM_BGK, B.LBM_F32, 128, 128, 128, tau=0.6)
    assert B.lbm_workspace_bytes(big) > B.LBM_NOALLOC_MAX_BYTES
    x = torch.zeros(16, device="cuda:0")
    with pytest.raises(B.LbmError) as e:
        B.lbm_step_noalloc(big, None, x.data_ptr(), x.data_ptr(), 1)
    assert e.value.code == B.LBM_EINVAL and "static maximum" in str(e.value) and str(B.LBM_NOALLOC_MAX_BYTES) in str(e.value)
    fits = B.make_params(B.LBM_D3Q19, B.LBM_BGK, B.LBM_F32, 64, 64, 64, tau=0.6)        # the documented limit case
    assert B.lbm_workspace_bytes(fits) <= B.LBM_NOALLOC_MAX_BYTES
    small = B.make_params(B.LBM_D3Q19, B.LBM_BGK, B.LBM_F32, 8, 8, 8, tau=0.6)
    with pytest.raises(B.LbmError) as e:
        B.lbm_step_noalloc(small, None, None, x.data_ptr(), 1)
    assert e.value.code == B.LBM_EINVAL
    aa = B.make_params(B.LBM_D3Q19, B.LBM_BGK, B.LBM_F32, 8, 8, 8, tau=0.6, store=B.LBM_STORE_AA)
    with pytest.raises(B.LbmError) as e:
        B.lbm_step_noalloc(aa, None, x.data_ptr(), x.data_ptr(), 1)
    assert e.value.code == B.LBM_EUNSUPPORTED
    bad = B.make_params(B.LBM_D3Q19, B.LBM_BGK, B.LBM_F32, 8, 8, 8, tau=0.4)
    with pytest.raises(B.LbmError) as e:
        B.lbm_step_noalloc(bad, None, x.data_ptr(), x.data_ptr(), 1)
    assert e.value.code == B.LBM_EINVAL and "tau" in str(e.value)
