"""The device functions of the default ("rx") kernel family, compiled for the host and run thread by thread
over bounds- and hazard-checked arrays (tests/host_emul/rx_emul.cu), against the fp64 oracle.  CPU only.

This is (i) a parity test of the kernel arithmetic that needs no GPU and (ii) the stand-in for
compute-sanitizer, which is closed on the GPU pool (profiles/r02_sanitizer.md): an out-of-bounds index, a
read of unwritten shared memory or a same-phase cross-thread hazard aborts the emulator with exit code 3.

Input file layout (little endian): int32 Nx,Ny,Nz,Nl,Nm,Ns,J,pad; float32 dkx,dky; complex64 G[s][m][l][z][kx][ky];
complex64 Phi[z][kx][ky]; float32 M[s][z][j][kx][ky]; float32 T[j][l]; float32 Tinv[l][j]; float32 (cos,sin)(2 pi t/Nx).
The tables are the oracle's fp64 values rounded once (reading R14)."""
import math
import os
import shutil
import subprocess

import numpy as np
import pytest

import gx_oracle as O
from paper_2209_06731_b200 import inputs as I

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "host_emul", "rx_emul.cu")
CSRC = os.path.join(HERE, "..", "paper_2209_06731_b200", "csrc")


@pytest.fixture(scope="module")
def emulator(tmp_path_factory):
    if shutil.which("nvcc") is None:
        pytest.skip("nvcc not available")
    exe = str(tmp_path_factory.mktemp("emul") / "rx_emul")
    deps = [SRC] + [os.path.join(CSRC, f) for f in ("nl_rx_kernels.cuh", "dft_packed.cuh", "dft_regs.cuh", "nl_kernels.cuh")]
    cache = os.path.join(HERE, "host_emul", "rx_emul.bin")          # git-ignored build product, reused when fresh
    if os.path.exists(cache) and all(os.path.getmtime(cache) > os.path.getmtime(d) for d in deps):
        return cache
    subprocess.check_call(["nvcc", "-O1", "-std=c++17", "-diag-suppress", "20011,20014", "-gencode",
                           "arch=compute_100a,code=sm_100a", "-o", exe, SRC])
    try:
        shutil.copy(exe, cache)
        return cache
    except OSError:
        return exe


def _run(emulator, tmp_path, cfg):
    geo = I.geometry_arrays(cfg)
    G = I.make_state(cfg, geo)
    Phi = O.field_solve(G, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species, tau_fac=cfg.tau_fac,
                        adiabatic=(cfg.Ns == 1)).astype(np.complex64)
    x, w, T, Tinv = O.laguerre_matrices(cfg.Nl)
    kx, ky = cfg.dkx * O.kx_index(cfg.Nx), cfg.dky * O.ky_index(cfg.Ny)
    kp2 = O.kperp2(kx, ky, geo["gds2"], geo["gds21"], geo["gds22"], cfg.shat)
    M = np.stack([O.gyro_table(O.b_species(kp2, geo["bmag"], sp.Z, sp.mass, sp.temp), x) for sp in cfg.species])
    t = 2.0 * math.pi * np.arange(cfg.Nx) / cfg.Nx
    tw = np.stack([np.cos(t), np.sin(t)], axis=1)
    fin, fout = str(tmp_path / "in.bin"), str(tmp_path / "out.bin")
    with open(fin, "wb") as f:
        f.write(np.array([cfg.Nx, cfg.Ny, cfg.Nz, cfg.Nl, cfg.Nm, cfg.Ns, len(x), 0], np.int32).tobytes())
        f.write(np.array([cfg.dkx, cfg.dky], np.float32).tobytes())
        for a, dt in [(G, np.complex64), (Phi, np.complex64), (M, np.float32), (T, np.float32), (Tinv, np.float32),
                      (tw, np.float32)]:
            f.write(np.ascontiguousarray(a, dtype=dt).tobytes())
    res = subprocess.run([emulator, fin, fout], capture_output=True, text=True)
    assert res.returncode == 0, res.stdout + res.stderr
    out = np.fromfile(fout, dtype=np.complex64).reshape(cfg.g_shape)
    ref = O.nonlinear_rhs(G, Phi, cfg.Nx, cfg.Ny, cfg.dkx, cfg.dky, cfg.shat, geo, cfg.species, method="dft")
    return out, ref


@pytest.mark.parametrize("Nx,Nz,Nl,Nm,Ns", [
    (64, 2, 3, 2, 1),       # J = 4, all planes in one staging chunk
    (64, 1, 6, 1, 2),       # J = 8, Nl > CAP: chunked staging; two species
    (192, 1, 4, 2, 1),      # the Cyclone plane (127 x 22 modes), J = 5
    (128, 1, 2, 1, 1),      # 128 = 8 x 16
])
def test_rx_family_on_the_host_matches_oracle(emulator, tmp_path, Nx, Nz, Nl, Nm, Ns):
    sp = [I.Species(), I.Species(Z=-1.0, mass=1.0 / 1836.0, amp=0.05)][:Ns]
    cfg = I.Config("emul", Nx, 64, Nz, Nl, Nm, sp, seed=4242 + Nx + Nl)
    out, ref = _run(emulator, tmp_path, cfg)
    assert np.all(np.isfinite(out))
    err = O.relative_max_error(out, ref)
    assert err <= 2e-5, err
    for l in range(Nl):
        assert O.relative_max_error(out[:, :, l], ref[:, :, l]) <= 2e-5, l
