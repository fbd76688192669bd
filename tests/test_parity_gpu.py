"""Parity of the CUDA path (through the C-ABI) against the fp64 oracle on the same seeded inputs.

Bar (BASELINE.json north_star): max|gpu - oracle| / max|oracle| <= 2e-5 per output array; index
maps, mask and (to fp64 rounding) the Gauss-Laguerre rule must match exactly."""
import numpy as np
import pytest

import gx_oracle as O
from paper_2209_06731_b200 import inputs as I

pytestmark = pytest.mark.gpu
TOL = 2e-5


@pytest.fixture(scope="module")
def torch_cuda():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _grid(cfg, geo):
    from paper_2209_06731_b200 import binding
    return binding.Grid(cfg, geo)


def _oracle_phi(cfg, geo, G):
    return O.field_solve(G, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species,
                         tau_fac=cfg.tau_fac, adiabatic=(cfg.Ns == 1)).astype(np.complex64)


def _gpu_nl(torch, grid, G, Phi):
    g = torch.from_numpy(G).cuda()
    phi = torch.from_numpy(Phi).cuda()
    out = torch.full_like(g, float("nan"))
    grid.nonlinear_rhs(g, phi, out)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def _oracle_nl(cfg, geo, G, Phi, **kw):
    return O.nonlinear_rhs(G, Phi, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species, **kw)


def test_maps_mask_and_quadrature_match_oracle(torch_cuda):
    for name in ["tiny", "cyclone", "hires", "w7x-shape"]:
        cfg = I.named_config(name)
        small = I.Config(name, cfg.Nx, cfg.Ny, 2, cfg.Nl, 1, cfg.species, geometry=cfg.geometry, seed=1)
        grid = _grid(small, I.geometry_arrays(small))
        m = grid.export_maps()
        assert np.array_equal(m["kx_index"], O.kx_index(cfg.Nx))
        assert np.array_equal(m["ky_index"], O.ky_index(cfg.Ny))
        assert np.array_equal(m["pad_row"], O.pad_row(cfg.Nx))
        assert np.array_equal(m["mask"], O.dealias_mask(cfg.Nx, cfg.Ny))
        x, w = O.gauss_laguerre(small.nj)
        assert np.allclose(m["lag_nodes"], x, rtol=1e-12, atol=0)
        assert np.allclose(m["lag_weights"], w, rtol=1e-10, atol=0)
        from paper_2209_06731_b200 import binding
        T, Tinv, M = binding.gx_export_tables(grid.h, small.Nl, small.Ns * 2 * small.nj * small.nakx * small.naky)
        _, _, To, Tinvo = O.laguerre_matrices(small.Nl)
        assert np.array_equal(T, To.astype(np.float32)) or np.max(np.abs(T - To)) <= 2e-7 * np.max(np.abs(To))
        assert np.max(np.abs(Tinv - Tinvo)) <= 2e-7 * np.max(np.abs(Tinvo))
        geo = grid.geo
        kx, ky = small.dkx * O.kx_index(cfg.Nx), small.dky * O.ky_index(cfg.Ny)
        sp = small.species[0]
        b = O.b_species(O.kperp2(kx, ky, geo["gds2"], geo["gds21"], geo["gds22"], small.shat), geo["bmag"],
                        sp.Z, sp.mass, sp.temp)
        Mo = O.gyro_table(b, x)                       # [z][j][kx][ky]
        Mg = M.reshape(small.Ns, 2, small.nj, small.nakx, small.naky)[0]
        assert np.max(np.abs(Mg - Mo)) < 1.5e-7
        grid.close()


def test_tiny_full_parity_against_definition(torch_cuda):
    cfg = I.named_config("tiny")
    geo = I.geometry_arrays(cfg)
    G = I.make_state(cfg, geo)
    Phi = _oracle_phi(cfg, geo, G)
    grid = _grid(cfg, geo)
    out = _gpu_nl(torch_cuda, grid, G, Phi)
    ref = _oracle_nl(cfg, geo, G, Phi, method="conv_c")        # the definition, every plane
    assert np.all(np.isfinite(out))
    assert O.relative_max_error(out, ref) <= TOL
    for l in range(cfg.Nl):                                   # per-l slabs too (stricter)
        assert O.relative_max_error(out[:, :, l], ref[:, :, l]) <= TOL
    # output properties that hold at any size
    K = (cfg.nakx - 1) // 2
    s = np.max(np.abs(ref))
    assert np.max(np.abs(out[..., cfg.nakx - 1:K:-1, 0] - np.conj(out[..., 1:K + 1, 0]))) < 1e-5 * s
    assert np.max(np.abs(out[..., 0, 0])) < 1e-5 * s
    grid.close()


def test_single_mode_closed_form_on_gpu(torch_cuda):
    # b = 0 (mass -> 0 gives M == 1), one chi mode, one g mode: exactly two output modes (oracle pin 4)
    cfg = I.Config("one", 16, 16, 2, 1, 1, [I.Species(mass=1e-30)], seed=3)
    geo = I.geometry_arrays(cfg)
    nakx, naky = cfg.nakx, cfg.naky
    G = np.zeros(cfg.g_shape, np.complex64)
    Phi = np.zeros(cfg.phi_shape, np.complex64)
    (pa, pb), (qa, qb) = (2, 1), (-1, 3)
    cp, gq = np.complex64(0.75 - 0.25j), np.complex64(-0.5 + 1.0j)
    Phi[:, pa, pb] = cp
    G[0, 0, 0, :, qa + nakx, qb] = gq
    grid = _grid(cfg, geo)
    out = _gpu_nl(torch_cuda, grid, G, Phi)
    cross = (cfg.dkx * pa) * (cfg.dky * qb) - (cfg.dky * pb) * (cfg.dkx * qa)
    expect = np.zeros_like(out, dtype=np.complex128)
    expect[0, 0, 0, :, pa + qa, pb + qb] = -cross * complex(cp) * complex(gq)
    expect[0, 0, 0, :, (qa - pa) + nakx, qb - pb] = cross * np.conj(complex(cp)) * complex(gq)
    assert np.max(np.abs(out - expect)) < 2e-6 * np.max(np.abs(expect))
    grid.close()


def test_cyclone_parity_full_array_and_sampled_definition(torch_cuda):
    cfg = I.named_config("cyclone")
    geo = I.geometry_arrays(cfg)
    G = I.make_state(cfg, geo)
    Phi = _oracle_phi(cfg, geo, G)
    grid = _grid(cfg, geo)
    out = _gpu_nl(torch_cuda, grid, G, Phi)
    assert np.all(np.isfinite(out))
    # full array against the pseudo-spectral oracle path (several tiles, ragged 127 x 22 planes)
    ref = _oracle_nl(cfg, geo, G, Phi, method="dft")
    err = O.relative_max_error(out, ref)
    assert err <= TOL, err
    for m in range(cfg.Nm):
        assert O.relative_max_error(out[:, m], ref[:, m]) <= TOL
    # sampled planes against the definition (direct convolution)
    planes = [(0, 0, 0), (0, 3, 11), (0, 7, 23)]
    refc = _oracle_nl(cfg, geo, G, Phi, method="conv_c", planes=planes)
    for (s, m, z) in planes:
        e = np.max(np.abs(out[s, m, :, z] - refc[s, m, :, z])) / np.max(np.abs(refc[s, m, :, z]))
        assert e <= TOL, (s, m, z, e)
    # free-energy invariant on the GPU result (holds at any size)
    W = O.free_energy_moment(G.astype(np.complex128), out.astype(np.complex128))
    scale = np.einsum("smlzxy->smz", np.abs(G.astype(np.complex128)) * np.abs(out))
    assert np.max(np.abs(W) / scale) < 2e-5
    grid.close()


@pytest.mark.parametrize("name,planes", [
    ("kinetic", [(0, 0, 0), (1, 0, 5), (1, 7, 31), (0, 4, 16)]),
    ("hires", [(0, 0, 0), (0, 15, 31), (0, 6, 9)]),
    ("stellarator", [(0, 0, 0), (0, 11, 127), (0, 5, 64)]),
    ("w7x-shape", [(0, 0, 0), (0, 7, 100)]),
])
def test_large_configs_sampled_planes(torch_cuda, name, planes):
    """Full-size runs in the bench's launch configuration; the oracle evaluates sampled (s,m,z) planes."""
    torch = torch_cuda
    cfg = I.named_config(name)
    geo = I.geometry_arrays(cfg)
    sm = sorted({(s, m) for (s, m, z) in planes} | {(s, 0) for s in range(cfg.Ns)})
    G = I.make_state(cfg, geo, planes=sm)           # only the sampled (s,m) slabs are non-zero
    Phi = _oracle_phi(cfg, geo, G)
    grid = _grid(cfg, geo)
    out = _gpu_nl(torch, grid, G, Phi)
    ref = _oracle_nl(cfg, geo, G, Phi, method="dft", planes=planes)
    for (s, m, z) in planes:
        a, r = out[s, m, :, z], ref[s, m, :, z]
        assert np.all(np.isfinite(a))
        e = np.max(np.abs(a - r)) / np.max(np.abs(r))
        assert e <= TOL, (name, s, m, z, e)
    # slabs that were zero on input must be exactly zero on output (bilinearity)
    zero_sm = [(s, m) for s in range(cfg.Ns) for m in range(cfg.Nm) if (s, m) not in sm]
    if zero_sm:
        s, m = zero_sm[0]
        assert np.all(out[s, m] == 0)
    grid.close()


@pytest.mark.parametrize("name", ["hires", "w7x-shape", "stellarator"])
def test_large_configs_full_array_all_slabs(torch_cuda, name):
    """BASELINE.json configs[3], [4] and the W7-X shape at full size, every (s,m,l,z) slab non-zero, in the
    launch configuration bench.py times, compared element by element with the pseudo-spectral oracle path
    (5-20 s of oracle time).  Two calls back to back on the same handle so that a cross-unit hazard (counter
    epoch, workspace slot reuse) would show as a difference between them."""
    torch = torch_cuda
    cfg = I.named_config(name)
    geo = I.geometry_arrays(cfg)
    G = I.make_state(cfg, geo)
    Phi = _oracle_phi(cfg, geo, G)
    grid = _grid(cfg, geo)
    g, phi = torch.from_numpy(G).cuda(), torch.from_numpy(Phi).cuda()
    out1 = torch.full_like(g, float("nan"))
    out2 = torch.full_like(g, float("nan"))
    grid.nonlinear_rhs(g, phi, out1)
    grid.nonlinear_rhs(g, phi, out2)
    torch.cuda.synchronize()
    assert torch.equal(out1, out2)
    out = out1.cpu().numpy()
    del out1, out2, g
    assert np.all(np.isfinite(out))
    ref = _oracle_nl(cfg, geo, G, Phi, method="dft")
    err = O.relative_max_error(out, ref)
    assert err <= TOL, (name, err)
    for l in range(cfg.Nl):
        e = O.relative_max_error(out[:, :, l], ref[:, :, l])
        assert e <= TOL, (name, "l", l, e)
    for m in range(cfg.Nm):
        e = O.relative_max_error(out[:, m], ref[:, m])
        assert e <= TOL, (name, "m", m, e)
    grid.close()


def test_zero_input_and_error_paths(torch_cuda):
    torch = torch_cuda
    from paper_2209_06731_b200 import binding as B
    cfg = I.named_config("tiny")
    grid = _grid(cfg, I.geometry_arrays(cfg))
    g = torch.zeros(cfg.g_shape, dtype=torch.complex64, device="cuda")
    phi = torch.zeros(cfg.phi_shape, dtype=torch.complex64, device="cuda")
    out = torch.full_like(g, float("nan"))
    grid.nonlinear_rhs(g, phi, out)
    torch.cuda.synchronize()
    assert torch.all(out == 0)
    with pytest.raises(B.GxError) as e:
        B.gx_nonlinear_rhs(grid.h, g.data_ptr(), phi.data_ptr(), g.data_ptr())
    assert e.value.code == B.GX_ERR_ARG
    with pytest.raises(B.GxError) as e:
        B.gx_nonlinear_rhs(grid.h, None, phi.data_ptr(), out.data_ptr())
    assert e.value.code == B.GX_ERR_ARG
    grid.close()
    for bad in [(15, 16), (16, 2), (16, 34)]:
        with pytest.raises(B.GxError) as e:
            B.gx_grid_create(bad[0], bad[1], 4, 2, 2, 1)
        assert e.value.code == B.GX_ERR_ARG
    with pytest.raises(B.GxError) as e:
        B.gx_grid_create(32, 32, 4, 2, 2, 1)       # valid size, no kernel instantiation
    assert e.value.code == B.GX_ERR_UNSUPPORTED
    h = B.gx_grid_create(16, 16, 4, 2, 2, 1)
    with pytest.raises(B.GxError) as e:
        B.gx_nonlinear_rhs(h, g.data_ptr(), phi.data_ptr(), out.data_ptr())
    assert e.value.code == B.GX_ERR_STATE
    B.gx_grid_destroy(h)


def test_compute_calls_refuse_stream_capture(torch_cuda):
    """The kernels take the call's epoch as an argument, so a caller's CUDA graph would replay stale epochs: the
    device compute calls return GX_ERR_STATE while their stream is capturing (and work again afterwards)."""
    torch = torch_cuda
    from paper_2209_06731_b200 import binding as B
    cfg = I.named_config("tiny")
    geo = I.geometry_arrays(cfg)
    G = I.make_state(cfg, geo)
    grid = _grid(cfg, geo)
    g = torch.from_numpy(G).cuda()
    phi = torch.from_numpy(_oracle_phi(cfg, geo, G)).cuda()
    out = torch.empty_like(g)
    grid.nonlinear_rhs(g, phi, out)
    torch.cuda.synchronize()
    ref = out.clone()
    side = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        graph.capture_begin()
        try:
            with pytest.raises(B.GxError) as e:
                grid.nonlinear_rhs(g, phi, out)
            assert e.value.code == B.GX_ERR_STATE
            phi.mul_(1.0)                       # something to record: an empty capture is an error of its own
        finally:
            graph.capture_end()
    torch.cuda.synchronize()
    out.zero_()
    grid.nonlinear_rhs(g, phi, out)
    torch.cuda.synchronize()
    assert torch.equal(out, ref)
    grid.close()


@pytest.mark.parametrize("name", ["tiny", "kinetic"])
def test_host_entry_point_matches_device_entry_point(torch_cuda, name):
    """gx_nonlinear_rhs_host pipelines Hermite blocks over three streams (two species: strided block copies);
    the result must be bit-identical to the one-shot device call, also when called twice in a row."""
    torch = torch_cuda
    cfg = I.named_config(name)
    geo = I.geometry_arrays(cfg)
    G = I.make_state(cfg, geo)
    Phi = _oracle_phi(cfg, geo, G)
    grid = _grid(cfg, geo)
    out_dev = _gpu_nl(torch, grid, G, Phi)
    gh, ph = torch.from_numpy(G).pin_memory(), torch.from_numpy(Phi).pin_memory()
    oh = torch.empty_like(gh).pin_memory()
    grid.nonlinear_rhs_host(gh, ph, oh)
    assert np.array_equal(oh.numpy(), out_dev)
    oh.zero_()
    grid.nonlinear_rhs_host(gh, ph, oh)
    assert np.array_equal(oh.numpy(), out_dev)
    assert np.array_equal(_gpu_nl(torch, grid, G, Phi), out_dev)      # and the device entry point still works after it
    grid.close()


def test_field_solve_parity(torch_cuda):
    """Boltzmann electrons (Eq. 6.1: tiny, cyclone) and two kinetic species (Eq. 4.23: kinetic)."""
    torch = torch_cuda
    for name in ["tiny", "cyclone", "kinetic"]:
        cfg = I.named_config(name)
        geo = I.geometry_arrays(cfg)
        G = I.make_state(cfg, geo, planes=[(s, 0) for s in range(cfg.Ns)])
        grid = _grid(cfg, geo)
        g = torch.from_numpy(G).cuda()
        phi = torch.empty(cfg.phi_shape, dtype=torch.complex64, device="cuda")
        grid.field_solve(g, phi)
        torch.cuda.synchronize()
        ref = O.field_solve(G, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species, tau_fac=cfg.tau_fac,
                            adiabatic=(cfg.Ns == 1))
        assert O.relative_max_error(phi.cpu().numpy(), ref) <= TOL, name
        if cfg.Ns == 2:     # the electron density really enters: the ion-only solve is a different potential
            ion_only = O.field_solve(G[:1], cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species[:1],
                                     adiabatic=False)
            assert O.relative_max_error(ion_only, ref) > 100 * TOL
        grid.close()


@pytest.mark.parametrize("family", ["scalar", "row", "rx", "rxp", "rxw"])
@pytest.mark.parametrize("name", ["tiny", "cyclone", "kinetic", "w7x-shape"])
def test_kernel_families_agree_with_oracle(torch_cuda, monkeypatch, family, name):
    """Every kernel family behind the C-ABI (GX_KERNELS, read at gx_grid_create) meets the same bar;
    a family without an instantiation for the grid falls through to the next one."""
    monkeypatch.setenv("GX_KERNELS", family)
    cfg = I.named_config(name)
    geo = I.geometry_arrays(cfg)
    planes = [(0, 0, 0), (cfg.Ns - 1, cfg.Nm - 1, cfg.Nz - 1), (0, cfg.Nm // 2, cfg.Nz // 3)]
    sm = sorted({(s, m) for (s, m, z) in planes} | {(s, 0) for s in range(cfg.Ns)})
    G = I.make_state(cfg, geo, planes=sm)
    Phi = _oracle_phi(cfg, geo, G)
    grid = _grid(cfg, geo)
    out = _gpu_nl(torch_cuda, grid, G, Phi)
    out2 = _gpu_nl(torch_cuda, grid, G, Phi)                 # second call: counters / staging reuse
    assert np.array_equal(out, out2)
    ref = _oracle_nl(cfg, geo, G, Phi, method="dft", planes=planes)
    for (s, m, z) in planes:
        a, r = out[s, m, :, z], ref[s, m, :, z]
        e = np.max(np.abs(a - r)) / np.max(np.abs(r))
        assert e <= TOL, (family, name, s, m, z, e)
    grid.close()


@pytest.mark.parametrize("Nx,Ny,family", [(48, 48, "scalar"), (96, 96, "scalar"), (128, 96, "scalar"), (192, 96, "scalar"),
                                          (96, 192, "scalar"), (96, 64, "row"), (64, 96, "row"), (64, 256, "row")])
def test_more_plane_shapes(torch_cuda, Nx, Ny, family):
    """Further (Nx, Ny) instantiations -- the paper's other perpendicular grids (Ny = 96 with Nx = 96 ... 192) and the
    transposed row configurations for Nx = 64 -- full array against the oracle, two species-free small batches."""
    cfg = I.Config(f"shape{Nx}x{Ny}", Nx, Ny, 3, 3, 2, [I.Species(tprim=6.9, fprim=2.2, nu_ss=0.01)], seed=I.BASE_SEED + 40 + Nx + Ny)
    geo = I.geometry_arrays(cfg)
    G = I.make_state(cfg, geo)
    Phi = _oracle_phi(cfg, geo, G)
    grid = _grid(cfg, geo)
    from paper_2209_06731_b200 import binding
    assert binding.FAMILY_NAMES[grid.query(binding.GX_Q_KERNEL_FAMILY)] == family
    out = _gpu_nl(torch_cuda, grid, G, Phi)
    out2 = _gpu_nl(torch_cuda, grid, G, Phi)
    assert np.array_equal(out, out2)
    ref = _oracle_nl(cfg, geo, G, Phi, method="dft")
    assert O.relative_max_error(out, ref) <= TOL, (Nx, Ny, O.relative_max_error(out, ref))
    for l in range(cfg.Nl):
        a, r = out[:, :, l], ref[:, :, l]
        assert np.max(np.abs(a - r)) <= TOL * np.max(np.abs(r)), (Nx, Ny, l)
    grid.close()


@pytest.mark.parametrize("name,cluster", [("cyclone", False), ("kinetic", False), ("nx64", False), ("small64", False), ("small192", False),
                                          ("cyclone", True), ("w7x-shape", True)])
def test_chained_calls_match_isolated_calls(torch_cuda, monkeypatch, name, cluster):
    """Consecutive gx_nonlinear_rhs calls on one stream overlap on the device (row family: the chi planes of call
    N+1 start under the tail of call N; dchi is double-buffered; bhat, out and the counters are reused across calls and
    ordered by flags, not by grid completion).  Eight back-to-back calls with DIFFERENT states and potentials, two of
    them writing the same output buffer, must give bit for bit what each call gives alone, and the oracle's result.
    (The transposed 64 x 192 configuration is covered by the w7x-shape case.)"""
    torch = torch_cuda
    if cluster:          # optional variant: a8 over the distributed shared memory of a J-CTA cluster (GX_CLUSTER, read per call)
        monkeypatch.setenv("GX_CLUSTER", "1")
    if name.startswith("small"):     # a handful of units: every SM sees the same chi planes again two calls later (L1 must not serve old lines)
        cfg = I.Config(name, int(name[5:]), 64, 2, 4, 2, [I.Species(tprim=6.9, fprim=2.2, nu_ss=0.01)], seed=I.BASE_SEED + 77)
    else:
        cfg = I.named_config(name)
    geo = I.geometry_arrays(cfg)
    sm = sorted({(s, m) for s in range(cfg.Ns) for m in (0, cfg.Nm // 2, cfg.Nm - 1)})
    G0 = I.make_state(cfg, geo, planes=sm)
    Phi0 = _oracle_phi(cfg, geo, G0)
    grid = _grid(cfg, geo)
    rng = np.random.default_rng(7)
    K = 8
    gs, phis = [], []
    for i in range(K):
        a, b = 1.0 + 0.25 * i, 1.0 - 0.1 * i
        gs.append(torch.from_numpy((a * G0).astype(np.complex64)).cuda())
        ph = (b * Phi0 * (1 + 0.05 * i * rng.standard_normal(Phi0.shape))).astype(np.complex64)
        ph[:, :, 0] = Phi0[:, :, 0] * b           # keep the ky = 0 column Hermitian
        phis.append(torch.from_numpy(ph).cuda())
    alone = []
    for i in range(K):                                        # each call by itself
        out = torch.full_like(gs[i], float("nan"))
        grid.nonlinear_rhs(gs[i], phis[i], out)
        torch.cuda.synchronize()
        alone.append(out.clone())
    outs = [torch.full_like(gs[0], float("nan")) for _ in range(K - 1)]
    for rep in range(25):                                     # back to back, no synchronisation in between: 200 calls
        for i in range(K):
            grid.nonlinear_rhs(gs[i], phis[i], outs[min(i, K - 2)])     # calls K-2 and K-1 share a buffer
            if i == K - 2:
                snap = outs[K - 2].clone()                    # stream-ordered copy between the two writers
        torch.cuda.synchronize()
        for i in range(K - 2):
            assert torch.equal(outs[i], alone[i]), (name, rep, i)
        assert torch.equal(snap, alone[K - 2]), (name, rep)
        assert torch.equal(outs[K - 2], alone[K - 1]), (name, rep)
        if rep % 5 == 4:                                      # vary the pattern: skip ahead by one input
            gs.append(gs.pop(0)); phis.append(phis.pop(0)); alone.append(alone.pop(0))
    alone = [a.cpu().numpy() for a in alone]
    planes = [(cfg.Ns - 1, cfg.Nm - 1, cfg.Nz - 1)]
    ref = _oracle_nl(cfg, geo, gs[3].cpu().numpy(), phis[3].cpu().numpy(), method="dft", planes=planes)     # (lists rotated together)
    for (s, m, z) in planes:
        a, r = alone[3][s, m, :, z], ref[s, m, :, z]
        assert np.max(np.abs(a - r)) / np.max(np.abs(r)) <= TOL
    grid.close()


def test_mixed_call_sequences_on_one_handle(torch_cuda):
    """Chained gx_nonlinear_rhs calls interleaved, without synchronisation, with gx_rhs (plain kernels + separate
    inverse-Laguerre kernel), the electromagnetic call, gx_field_solve and the host entry point: every result equals
    the one the same call gives alone (the counters' epochs and the two dchi buffers survive every transition)."""
    torch = torch_cuda
    cfg = I.named_config("cyclone")
    geo = I.geometry_arrays(cfg)
    sm = sorted({(0, m) for m in (0, 1, cfg.Nm - 1)})
    G0 = I.make_state(cfg, geo, planes=sm)
    grid = _grid(cfg, geo)
    gs = [torch.from_numpy(((1.0 + 0.3 * i) * G0).astype(np.complex64)).cuda() for i in range(4)]
    phis = [torch.empty(cfg.phi_shape, dtype=torch.complex64, device="cuda") for _ in range(4)]
    for i in range(4):
        grid.field_solve(gs[i], phis[i])
    zero = torch.zeros_like(phis[0])
    gh = gs[2].cpu().pin_memory(); ph = phis[2].cpu().pin_memory()
    ops = ["nl", "nl", "rhs", "nl", "em", "nl", "rhs", "rhs", "nl", "host", "nl", "nl"]

    def run(k, op, out):
        i = k % 4
        if op == "nl":
            grid.nonlinear_rhs(gs[i], phis[i], out)
        elif op == "rhs":
            grid.rhs(gs[i], out)
        elif op == "em":
            grid.nonlinear_rhs_em(gs[i], phis[i], zero, zero, out)
        else:
            oh = torch.empty_like(gh).pin_memory()
            grid.nonlinear_rhs_host(gh, ph, oh)
            out.copy_(oh, non_blocking=False)

    alone = []
    for k, op in enumerate(ops):
        out = torch.full_like(gs[0], float("nan"))
        run(k, op, out)
        torch.cuda.synchronize()
        alone.append(out.cpu().numpy())
    assert np.array_equal(alone[4], alone[0])             # apar = bpar = 0: the electromagnetic call is the electrostatic one
    for rep in range(2):
        outs = [torch.full_like(gs[0], float("nan")) for _ in ops]
        for k, op in enumerate(ops):
            run(k, op, outs[k])
        torch.cuda.synchronize()
        for k, op in enumerate(ops):
            assert np.array_equal(outs[k].cpu().numpy(), alone[k]), (rep, k, op)
    grid.close()


# ------------------------------------------------------------------------------------------------
# linear terms and the full right-hand side against oracle/gx_linear.py
import gx_linear as OL


def _oracle_lin(cfg, geo, G, Phi):
    return OL.linear_rhs(G, Phi, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species)


@pytest.mark.parametrize("point", ["march", "stencil"])
@pytest.mark.parametrize("name", ["tiny", "cyclone", "kinetic", "w7x-shape"])
def test_linear_rhs_parity(torch_cuda, monkeypatch, name, point):
    """point: the pointwise terms by the marching kernel (default) or by the per-(s,m) stencil kernel (GX_LIN_POINT)."""
    torch = torch_cuda
    if point == "stencil":
        monkeypatch.setenv("GX_LIN_POINT", "stencil")
    cfg = I.named_config(name)
    if name == "w7x-shape":
        cfg = I.Config(cfg.name, cfg.Nx, cfg.Ny, cfg.Nz, cfg.Nl, 4, cfg.species, geometry=cfg.geometry, seed=cfg.seed)
    geo = I.geometry_arrays(cfg)
    G = I.make_state(cfg, geo)
    Phi = _oracle_phi(cfg, geo, G)
    grid = _grid(cfg, geo)
    g, phi = torch.from_numpy(G).cuda(), torch.from_numpy(Phi).cuda()
    out = torch.full_like(g, float("nan"))
    grid.linear_rhs(g, phi, out)
    torch.cuda.synchronize()
    out = out.cpu().numpy()
    ref = _oracle_lin(cfg, geo, G, Phi)
    assert np.all(np.isfinite(out))
    assert O.relative_max_error(out, ref) <= TOL
    for s in range(cfg.Ns):
        for m in range(cfg.Nm):                                # per-(s,m) slabs: every stencil row is exercised
            assert O.relative_max_error(out[s, m], ref[s, m]) <= 5 * TOL, (s, m)
    grid.close()


@pytest.mark.parametrize("name", ["tiny", "cyclone", "kinetic"])
def test_full_rhs_parity(torch_cuda, name):
    """gx_rhs = field solve + (-N) + linear terms, all on the device, against the oracle's rhs()."""
    torch = torch_cuda
    cfg = I.named_config(name)
    geo = I.geometry_arrays(cfg)
    G = I.make_state(cfg, geo)
    grid = _grid(cfg, geo)
    g = torch.from_numpy(G).cuda()
    out = torch.full_like(g, float("nan"))
    grid.rhs(g, out)
    torch.cuda.synchronize()
    out = out.cpu().numpy()
    ref = OL.rhs(G, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species, tau_fac=cfg.tau_fac)
    assert np.all(np.isfinite(out))
    assert O.relative_max_error(out, ref) <= TOL
    for s_ in range(cfg.Ns):                                   # per species (the electron slabs are much larger)
        assert O.relative_max_error(out[s_], ref[s_]) <= TOL, s_
    # the nonlinear part alone must still be visible at this tolerance (it is not drowned by the linear part)
    lin = OL.rhs(G, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species, tau_fac=cfg.tau_fac, nonlinear=False)
    assert O.relative_max_error(lin, ref) > 10 * TOL
    grid.close()


def test_ssprk3_steps_parity(torch_cuda):
    """two SSP-RK3 steps of gx_rhs on the tiny flux tube against the oracle's stepper."""
    torch = torch_cuda
    cfg = I.named_config("tiny")
    geo = I.geometry_arrays(cfg)
    G = I.make_state(cfg, geo)
    grid = _grid(cfg, geo)
    g = torch.from_numpy(G).cuda()
    dt = 0.02
    f = lambda y: OL.rhs(y, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species, tau_fac=cfg.tau_fac)
    ref = G.astype(np.complex128)
    for _ in range(2):
        grid.ssprk3_step(g, dt)
        ref = OL.ssp_rk3_step(ref, dt, f)
    torch.cuda.synchronize()
    out = g.cpu().numpy()
    assert np.all(np.isfinite(out))
    assert O.relative_max_error(out, ref) <= TOL
    assert O.relative_max_error(G, ref) > 100 * TOL          # the state really moved
    grid.close()


def test_ssprk3_one_step_parity_cyclone(torch_cuda):
    """One SSP-RK3 step of gx_rhs at the Cyclone size (three device field solves, nonlinear and linear terms,
    fused stage kernels) against the oracle's stepper."""
    torch = torch_cuda
    cfg = I.named_config("cyclone")
    geo = I.geometry_arrays(cfg)
    G = I.make_state(cfg, geo)
    grid = _grid(cfg, geo)
    g = torch.from_numpy(G).cuda()
    dt = 0.01
    grid.ssprk3_step(g, dt)
    torch.cuda.synchronize()
    out = g.cpu().numpy()
    f = lambda y: OL.rhs(y, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species, tau_fac=cfg.tau_fac)
    ref = OL.ssp_rk3_step(G.astype(np.complex128), dt, f)
    assert np.all(np.isfinite(out))
    assert O.relative_max_error(out, ref) <= TOL
    assert O.relative_max_error(out - G, ref - G) <= 50 * TOL     # the increment itself, not just the state
    grid.close()


@pytest.mark.parametrize("name", ["tiny", "kinetic"])
def test_full_rhs_parity_with_twist_shift_linking(torch_cuda, name):
    """gx_rhs with gx_boundary_set(1): device field solve + nonlinear term + linked linear terms."""
    torch = torch_cuda
    from paper_2209_06731_b200 import binding
    cfg = I.named_config(name)
    geo = I.geometry_arrays(cfg)
    G = I.make_state(cfg, geo)
    grid = binding.Grid(cfg, geo, linked=True)
    g = torch.from_numpy(G).cuda()
    out = torch.full_like(g, float("nan"))
    grid.rhs(g, out)
    torch.cuda.synchronize()
    out = out.cpu().numpy()
    ref = OL.rhs(G, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species, tau_fac=cfg.tau_fac,
                 boundary="linked")
    assert np.all(np.isfinite(out))
    assert O.relative_max_error(out, ref) <= TOL
    grid.close()


@pytest.mark.parametrize("Nx,Ny,Nz,Nl,Nm,Ns", [
    (64, 64, 3, 1, 1, 1),      # one Laguerre moment (J = 1), one Hermite moment, odd Nz: degenerate batch sizes
    (64, 64, 2, 3, 2, 2),      # J = 4, two species on the row family
    (128, 64, 2, 4, 3, 1),     # odd Nm
    (256, 64, 1, 2, 2, 1),     # NX = 256 (scalar family), single z
    (16, 16, 1, 5, 1, 1),      # Nl = 5 -> J = 7 on the smallest plane
])
def test_degenerate_and_ragged_shapes(torch_cuda, Nx, Ny, Nz, Nl, Nm, Ns):
    """Edge shapes through the default kernel family: every (s,m,z) plane against the pseudo-spectral oracle."""
    sp = [I.Species(), I.Species(Z=-1.0, mass=1.0 / 1836.0, amp=0.05)][:Ns]
    cfg = I.Config("edge", Nx, Ny, Nz, Nl, Nm, sp, seed=777 + Nx + Nl)
    geo = I.geometry_arrays(cfg)
    G = I.make_state(cfg, geo)
    Phi = _oracle_phi(cfg, geo, G)
    grid = _grid(cfg, geo)
    out = _gpu_nl(torch_cuda, grid, G, Phi)
    ref = _oracle_nl(cfg, geo, G, Phi, method="dft")
    assert np.all(np.isfinite(out))
    assert O.relative_max_error(out, ref) <= TOL
    grid.close()


def test_calls_on_a_side_stream_and_interleaved_grids(torch_cuda):
    """Two handles used alternately on a non-default stream: per-handle counters and workspaces do not interfere."""
    torch = torch_cuda
    cfgs = [I.named_config("tiny"), I.Config("b", 64, 64, 2, 2, 2, [I.Species()], seed=5)]
    st = torch.cuda.Stream()
    items = []
    for cfg in cfgs:
        geo = I.geometry_arrays(cfg)
        G = I.make_state(cfg, geo)
        Phi = _oracle_phi(cfg, geo, G)
        items.append((cfg, geo, G, Phi, _grid(cfg, geo)))
    outs = []
    with torch.cuda.stream(st):
        bufs = [(torch.from_numpy(G).cuda(), torch.from_numpy(Phi).cuda()) for (_, _, G, Phi, _) in items]
        for rep in range(3):
            for (cfg, geo, G, Phi, grid), (g, phi) in zip(items, bufs):
                out = torch.full_like(g, float("nan"))
                grid.nonlinear_rhs(g, phi, out)
                if rep == 2:
                    outs.append(out)
    st.synchronize()
    for (cfg, geo, G, Phi, grid), out in zip(items, outs):
        ref = _oracle_nl(cfg, geo, G, Phi, method="dft")
        assert O.relative_max_error(out.cpu().numpy(), ref) <= TOL
        grid.close()


@pytest.mark.parametrize("name,zlink", [("tiny", "spectral"), ("cyclone", "spectral"), ("kinetic", "spectral"), ("cyclone", "dense")])
def test_linear_rhs_parity_with_twist_shift_linking(torch_cuda, monkeypatch, name, zlink):
    """gx_boundary_set(1): the z operators act on the linked extended domains of Eq. 4.29.  Chains of more
    than four links go through the harmonics of the extended domain (default) or through circulant products (GX_ZLINK=dense)."""
    torch = torch_cuda
    if zlink == "dense":
        monkeypatch.setenv("GX_ZLINK", "dense")
    from paper_2209_06731_b200 import binding
    cfg = I.named_config(name)
    geo = I.geometry_arrays(cfg)
    G = I.make_state(cfg, geo)
    Phi = _oracle_phi(cfg, geo, G)
    grid = binding.Grid(cfg, geo, linked=True)
    g, phi = torch.from_numpy(G).cuda(), torch.from_numpy(Phi).cuda()
    out = torch.full_like(g, float("nan"))
    grid.linear_rhs(g, phi, out)
    torch.cuda.synchronize()
    out = out.cpu().numpy()
    ref = OL.linear_rhs(G, Phi, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species, boundary="linked")
    per = OL.linear_rhs(G, Phi, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species, boundary="periodic")
    assert np.all(np.isfinite(out))
    assert O.relative_max_error(out, ref) <= TOL
    assert O.relative_max_error(per, ref) > 100 * TOL           # the linking really changes the answer
    for s in range(cfg.Ns):
        for m in range(cfg.Nm):
            assert O.relative_max_error(out[s, m], ref[s, m]) <= 5 * TOL, (s, m)
    grid.close()


def test_linked_boundary_needs_a_quantised_box(torch_cuda):
    from paper_2209_06731_b200 import binding as B
    cfg = I.named_config("tiny")
    geo = I.geometry_arrays(cfg)
    h = B.gx_grid_create(cfg.Nx, cfg.Ny, cfg.Nz, cfg.Nl, cfg.Nm, 1)
    B.gx_box_set(h, cfg.dky, 1.0123 * cfg.dkx, cfg.shat)
    B.gx_species_set(h, 0, 1.0, 1.0, 1.0, 1.0)
    B.gx_boundary_set(h, 1)
    with pytest.raises(B.GxError) as e:
        B.gx_geometry_set(h, geo["bmag"], geo["gds2"], geo["gds21"], geo["gds22"], geo["gbdrift"], geo["gbdrift0"],
                          geo["cvdrift"], geo["cvdrift0"], geo["bgrad"], geo["jacobian"], geo["gradpar"])
    assert e.value.code == B.GX_ERR_ARG
    B.gx_grid_destroy(h)


@pytest.mark.parametrize("name,linked", [("tiny", False), ("tiny", True), ("cyclone", True), ("hires", False)])
def test_linear_rhs_parity_with_end_damping(torch_cuda, name, linked):
    """Eq. 4.30: the wave-absorbing end layer on periodic and on linked extended domains
    (split pointwise kernel for Nl <= 4, generic kernel for hires with Nl = 8)."""
    torch = torch_cuda
    from paper_2209_06731_b200 import binding
    cfg = I.named_config(name)
    if name == "hires":
        cfg = I.Config(cfg.name, cfg.Nx, cfg.Ny, 8, cfg.Nl, 4, cfg.species, decay=cfg.decay, seed=cfg.seed)
    geo = I.geometry_arrays(cfg)
    G = I.make_state(cfg, geo)
    Phi = _oracle_phi(cfg, geo, G)
    dmp = dict(A=0.8, width_frac=0.125)
    grid = binding.Grid(cfg, geo, linked=linked, damping=dmp)
    g, phi = torch.from_numpy(G).cuda(), torch.from_numpy(Phi).cuda()
    out = torch.full_like(g, float("nan"))
    grid.linear_rhs(g, phi, out)
    torch.cuda.synchronize()
    out = out.cpu().numpy()
    bc = "linked" if linked else "periodic"
    ref = OL.linear_rhs(G, Phi, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species, boundary=bc, damping=dmp)
    off = OL.linear_rhs(G, Phi, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species, boundary=bc)
    assert np.all(np.isfinite(out))
    assert O.relative_max_error(out, ref) <= TOL
    assert O.relative_max_error(off, ref) > 20 * TOL           # the layer is visible at this tolerance
    grid.close()


# ------------------------------------------------------------------------------------------------
# electromagnetic brackets and field solve
@pytest.mark.parametrize("name", ["tiny", "kinetic"])
def test_em_nonlinear_rhs_parity(torch_cuda, name):
    """gx_nonlinear_rhs_em against the oracle's nonlinear_rhs_em (App. D Eq. D1 lines 1-4): every plane on tiny,
    sampled planes at the kinetic size; each of the three potentials is visible on its own at the tolerance."""
    torch = torch_cuda
    cfg = I.named_config(name)
    geo = I.geometry_arrays(cfg)
    G = I.make_state(cfg, geo)
    Phi = _oracle_phi(cfg, geo, G)
    Apar = (0.7 * I.random_phi(cfg, geo, seed_offset=101)).astype(np.complex64)
    Bpar = (0.4 * I.random_phi(cfg, geo, seed_offset=202)).astype(np.complex64)
    grid = _grid(cfg, geo)
    g = torch.from_numpy(G).cuda()
    f = [torch.from_numpy(a).cuda() for a in (Phi, Apar, Bpar)]
    out = torch.full_like(g, float("nan"))
    grid.nonlinear_rhs_em(g, f[0], f[1], f[2], out)
    torch.cuda.synchronize()
    out = out.cpu().numpy()
    planes = None if name == "tiny" else [(0, 0, 0), (1, 0, 5), (1, 7, 31), (0, 4, 16), (1, 3, 9)]
    kw = dict(method="dft", planes=planes)
    ref = O.nonlinear_rhs_em(G, Phi, Apar, Bpar, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species, **kw)
    es = O.nonlinear_rhs(G, Phi, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species, **kw)
    noA = O.nonlinear_rhs_em(G, Phi, 0 * Apar, Bpar, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species, **kw)
    sel = [(s, m, z) for s in range(cfg.Ns) for m in range(cfg.Nm) for z in range(cfg.Nz)] if planes is None else planes
    assert np.all(np.isfinite(out))
    for (s, m, z) in sel:
        a, r = out[s, m, :, z], ref[s, m, :, z]
        den = np.max(np.abs(r))
        assert np.max(np.abs(a - r)) <= TOL * den, (s, m, z)
    big = max(np.max(np.abs(ref[s, m, :, z])) for (s, m, z) in sel)
    assert max(np.max(np.abs((es - ref)[s, m, :, z])) for (s, m, z) in sel) > 100 * TOL * big
    assert max(np.max(np.abs((noA - ref)[s, m, :, z])) for (s, m, z) in sel) > 100 * TOL * big
    assert max(np.max(np.abs((noA - es)[s, m, :, z])) for (s, m, z) in sel) > 100 * TOL * big
    # zero vector potentials: the electrostatic entry point, bit for bit
    zero = torch.zeros_like(f[0])
    out0 = torch.full_like(g, float("nan"))
    grid.nonlinear_rhs_em(g, f[0], zero, zero, out0)
    torch.cuda.synchronize()
    assert np.array_equal(out0.cpu().numpy(), _gpu_nl(torch, grid, G, Phi))
    grid.close()


def test_em_field_solve_parity(torch_cuda):
    torch = torch_cuda
    cfg = I.named_config("kinetic")
    geo = I.geometry_arrays(cfg)
    G = I.make_state(cfg, geo, planes=[(s, m) for s in range(cfg.Ns) for m in (0, 1)])
    grid = _grid(cfg, geo)
    g = torch.from_numpy(G).cuda()
    f = [torch.empty(cfg.phi_shape, dtype=torch.complex64, device="cuda") for _ in range(3)]
    for beta in (0.0, 0.01):
        grid.field_solve_em(g, beta, f[0], f[1], f[2])
        torch.cuda.synchronize()
        ref = O.field_solve_em(G, beta, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species)
        for a, r, nm in zip(f, ref, ("phi", "apar", "bpar")):
            if np.max(np.abs(r)) == 0:
                assert torch.all(a == 0), nm
            else:
                assert O.relative_max_error(a.cpu().numpy(), r) <= TOL, (beta, nm)
    grid.close()


@pytest.mark.parametrize("Nz,Nl,Nm", [(64, 6, 5), (96, 2, 4), (128, 6, 4), (128, 4, 5)])
def test_linear_rhs_parity_z_fft_path(torch_cuda, Nz, Nl, Nm):
    """Long field lines (Nz = 64, 96, 128): the parallel derivative and |k_par| by FFT in z (Eq. 4.10-4.11)
    instead of circulant products, in the fused kernel (Nl > 4) and behind the pointwise kernel (Nl <= 4)."""
    torch = torch_cuda
    cfg = I.Config("zfft", 16, 16, Nz, Nl, Nm, [I.Species(tprim=3.0, fprim=1.0, nu_ss=0.01)], geometry="harmonics", seed=900 + Nz + Nl)
    geo = I.geometry_arrays(cfg)
    G = I.make_state(cfg, geo)
    Phi = _oracle_phi(cfg, geo, G)
    grid = _grid(cfg, geo)
    g, phi = torch.from_numpy(G).cuda(), torch.from_numpy(Phi).cuda()
    out = torch.full_like(g, float("nan"))
    grid.linear_rhs(g, phi, out)
    torch.cuda.synchronize()
    out = out.cpu().numpy()
    ref = _oracle_lin(cfg, geo, G, Phi)
    assert np.all(np.isfinite(out))
    assert O.relative_max_error(out, ref) <= TOL
    for m in range(cfg.Nm):
        assert O.relative_max_error(out[0, m], ref[0, m]) <= 5 * TOL, m
    # accumulate form (gx_rhs) through the same kernels
    out2 = torch.full_like(g, float("nan"))
    grid.rhs(g, out2)
    torch.cuda.synchronize()
    ref2 = OL.rhs(G, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species, tau_fac=cfg.tau_fac)
    assert O.relative_max_error(out2.cpu().numpy(), ref2) <= TOL
    grid.close()
