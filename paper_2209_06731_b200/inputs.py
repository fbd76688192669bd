"""Seeded synthetic inputs for the nonlinear E×B hot path.

This module serves BOTH the CUDA path and the oracle and therefore holds none of the
method's arithmetic: no Laguerre quadrature, no Bessel functions, no FFT, no bracket.
It only produces the *data* the C-ABI calls take: box parameters, per-z geometry
coefficient arrays (Eq. E4-E11 name them), species parameters and
a seeded spectral state ``g`` in the layout ``[s][m][l][z][kx][ky]``.

Random numbers come from a counter-based generator (splitmix64 of ``seed`` and a flat
element counter, then Box-Muller), so any slice of any configuration can be regenerated
without materialising the rest, and so nothing depends on a library RNG's stream order.

The five named configurations are the ones in BASELINE.json ``configs`` (shapes from
PAPER.md lines 804-826, App. G).  They stand in for the paper's Cyclone-base-case and W7-X
runs, whose equilibria and turbulent states are not available here.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

BASE_SEED = 22090673

_U64 = np.uint64
_MASK53 = (1 << 53) - 1


# ----------------------------------------------------------------------------- sizes
def dealiased_counts(Nx: int, Ny: int) -> tuple[int, int]:
    """(nakx, naky) of the 2/3-rule sets; reproduces 192->127, 64->22, 64->43, 192->64
     and 16->11, 16->6 (BASELINE.json configs[0])."""
    return 1 + 2 * ((Nx - 1) // 3), 1 + (Ny - 1) // 3


def num_mu_nodes(Nl: int) -> int:
    """J = floor((3*Nl-1)/2) Gauss-Laguerre nodes (reading R2)."""
    return (3 * Nl - 1) // 2


# ----------------------------------------------------------------------------- config
@dataclass
class Species:
    Z: float = 1.0
    mass: float = 1.0
    temp: float = 1.0   # tau_s
    dens: float = 1.0
    tprim: float = 0.0  # R/L_T
    fprim: float = 0.0  # R/L_n
    nu_ss: float = 0.0
    amp: float = 1.0    # amplitude factor of the synthetic g (not a library parameter)


@dataclass
class Config:
    name: str
    Nx: int
    Ny: int
    Nz: int
    Nl: int
    Nm: int
    species: list = field(default_factory=lambda: [Species()])
    dky: float = 0.1
    shat: float = 0.8
    q: float = 1.4
    eps: float = 0.18
    geometry: str = "s-alpha"      # or "harmonics"
    decay: float = 2.0             # moment decay r in r^-(l+m)
    tau_fac: float = 1.0           # adiabatic-electron T_i/T_e (used when one species)
    seed: int = BASE_SEED

    @property
    def Ns(self) -> int:
        return len(self.species)

    @property
    def nakx(self) -> int:
        return dealiased_counts(self.Nx, self.Ny)[0]

    @property
    def naky(self) -> int:
        return dealiased_counts(self.Nx, self.Ny)[1]

    @property
    def nj(self) -> int:
        return num_mu_nodes(self.Nl)

    @property
    def dkx(self) -> float:
        """Twist-and-shift box: Lx/Ly = jtwist/(2 pi |shat|)."""
        jtwist = max(1, int(round(2.0 * math.pi * abs(self.shat))))
        return 2.0 * math.pi * abs(self.shat) * self.dky / jtwist

    @property
    def g_shape(self) -> tuple:
        return (self.Ns, self.Nm, self.Nl, self.Nz, self.nakx, self.naky)

    @property
    def phi_shape(self) -> tuple:
        return (self.Nz, self.nakx, self.naky)

    @property
    def grid_point_moments(self) -> int:
        return self.Nx * self.Ny * self.Nz * self.Nl * self.Nm * self.Ns


def named_config(name: str) -> Config:
    ion = dict(Z=1.0, mass=1.0, temp=1.0, dens=1.0)
    if name == "tiny":
        return Config("tiny", 16, 16, 8, 2, 4, [Species(**ion, tprim=6.9, fprim=2.2, nu_ss=0.01)],
                      seed=BASE_SEED + 0)
    if name == "cyclone":
        return Config("cyclone", 192, 64, 24, 4, 8, [Species(**ion, tprim=6.9, fprim=2.2, nu_ss=0.01)],
                      seed=BASE_SEED + 1)
    if name == "kinetic":
        me = 1.0 / 1836.0
        return Config("kinetic", 128, 64, 32, 4, 8,
                      [Species(**ion, tprim=6.9, fprim=2.2, nu_ss=1.65e-4),
                       Species(Z=-1.0, mass=me, temp=1.0, dens=1.0, tprim=6.9, fprim=2.2,
                               nu_ss=0.01, amp=math.sqrt(me))],
                      seed=BASE_SEED + 2)
    if name == "hires":
        return Config("hires", 256, 96, 32, 8, 16, [Species(**ion, tprim=6.9, fprim=2.2, nu_ss=0.01)],
                      decay=1.3, seed=BASE_SEED + 3)
    if name == "stellarator":
        return Config("stellarator", 192, 192, 128, 6, 12,
                      [Species(**ion, tprim=3.0, fprim=1.0, nu_ss=0.01)],
                      geometry="harmonics", seed=BASE_SEED + 4)
    if name == "w7x-shape":   # the paper's own W7-X grid, SURVEY row f3
        return Config("w7x-shape", 64, 192, 128, 4, 8,
                      [Species(**ion, tprim=3.0, fprim=1.0, nu_ss=0.01)],
                      geometry="harmonics", seed=BASE_SEED + 5)
    if name.startswith("nx") and name[2:].isdigit():   # Nx sweep at the Cyclone velocity/parallel resolution (cf. Fig. 10)
        return Config(name, int(name[2:]), 64, 24, 4, 8, [Species(**ion, tprim=6.9, fprim=2.2, nu_ss=0.01)],
                      seed=BASE_SEED + 6)
    raise KeyError(name)


CONFIG_NAMES = ["tiny", "cyclone", "kinetic", "hires", "stellarator"]


# ----------------------------------------------------------------------------- index sets
def kx_integers(Nx: int) -> np.ndarray:
    """Compact kx integers in FFT order 0..K,-K..-1."""
    nakx, _ = dealiased_counts(Nx, 4)
    K = (nakx - 1) // 2
    return np.concatenate([np.arange(0, K + 1), np.arange(-K, 0)]).astype(np.int64)


def ky_integers(Ny: int) -> np.ndarray:
    _, naky = dealiased_counts(4, Ny)
    return np.arange(naky, dtype=np.int64)


# ----------------------------------------------------------------------------- geometry
def z_grid(Nz: int) -> np.ndarray:
    return -math.pi + 2.0 * math.pi * np.arange(Nz) / Nz


def geometry_arrays(cfg: Config) -> dict:
    """Per-z coefficient arrays (float64, length Nz) plus the constant ``gradpar``.

    "s-alpha": textbook circular s-alpha model with alpha_MHD = 0, lengths normalised to R.
    "harmonics": seeded sums of 8 integer harmonics about a mean (BASELINE.json configs[4]);
    the metric is built from a Cholesky factor so that k_perp^2 >= 0 by construction.
    """
    z = z_grid(cfg.Nz)
    sh = cfg.shat
    if cfg.geometry == "s-alpha":
        bmag = 1.0 / (1.0 + cfg.eps * np.cos(z))
        gradpar = 1.0 / cfg.q
        gds2 = 1.0 + (sh * z) ** 2
        gds21 = -sh * (sh * z)
        gds22 = np.full_like(z, sh * sh)
        gbdrift = 2.0 * (np.cos(z) + sh * z * np.sin(z))
        cvdrift = gbdrift.copy()
        gbdrift0 = -2.0 * sh * np.sin(z)
        cvdrift0 = gbdrift0.copy()
        bgrad = gradpar * cfg.eps * np.sin(z) / (1.0 + cfg.eps * np.cos(z))  # grad_par ln B
    elif cfg.geometry == "harmonics":
        rng = np.random.default_rng(cfg.seed ^ 0x5EED)

        def series(mean):
            a = 0.2 * rng.uniform(-1.0, 1.0, 8) / np.arange(1, 9)
            ph = rng.uniform(0.0, 2.0 * math.pi, 8)
            s = sum(a[h] * np.cos((h + 1) * z + ph[h]) for h in range(8))
            return mean * (1.0 + s) if mean != 0.0 else s

        bmag = series(1.0)
        A = series(1.0)
        C = series(1.0)
        D = series(0.0)
        gradpar = 1.0 / cfg.q
        gds22 = sh * sh * A * A
        gds21 = sh * A * D
        gds2 = C * C + D * D
        gbdrift = series(1.0)
        cvdrift = series(1.0)
        gbdrift0 = series(0.0)
        cvdrift0 = gbdrift0.copy()
        # grad_par ln B by spectral differentiation of ln(bmag) (2 pi periodic, integer harmonics)
        lnb = np.log(bmag)
        kz = np.fft.fftfreq(cfg.Nz, d=1.0 / cfg.Nz)
        if cfg.Nz % 2 == 0:
            kz[cfg.Nz // 2] = 0.0
        bgrad = gradpar * np.real(np.fft.ifft(1j * kz * np.fft.fft(lnb)))
    else:
        raise ValueError(cfg.geometry)
    jacobian = 1.0 / (gradpar * bmag)
    return dict(z=z, bmag=bmag, gds2=gds2, gds21=gds21, gds22=gds22, gbdrift=gbdrift,
                gbdrift0=gbdrift0, cvdrift=cvdrift, cvdrift0=cvdrift0, bgrad=bgrad,
                jacobian=jacobian, gradpar=float(gradpar))


# ----------------------------------------------------------------------------- RNG
def _splitmix64(x: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):
        x = (x + _U64(0x9E3779B97F4A7C15))
        x = (x ^ (x >> _U64(30))) * _U64(0xBF58476D1CE4E5B9)
        x = (x ^ (x >> _U64(27))) * _U64(0x94D049BB133111EB)
        x = x ^ (x >> _U64(31))
    return x


def counter_normals(seed: int, start: int, count: int) -> np.ndarray:
    """Standard normals n(start) .. n(start+count-1) of the stream ``seed``.

    n(c) = sqrt(-2 ln u1) cos(2 pi u2) with (u1,u2) from splitmix64 of the counter 2c, 2c+1
    offset by a hash of the seed; u in (0,1] / [0,1).
    """
    c = np.arange(start, start + count, dtype=np.uint64)
    with np.errstate(over="ignore"):
        base = _splitmix64(np.array([seed], dtype=np.uint64))[0]
        h1 = _splitmix64(base + _U64(2) * c)
        h2 = _splitmix64(base + _U64(2) * c + _U64(1))
    u1 = ((h1 >> _U64(11)).astype(np.float64) + 1.0) / float(1 << 53)   # (0,1]
    u2 = (h2 >> _U64(11)).astype(np.float64) / float(1 << 53)           # [0,1)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * math.pi * u2)


# ----------------------------------------------------------------------------- state
def _envelope(cfg: Config, geo: dict) -> np.ndarray:
    """(1 + k_perp^2)^-1 on [z][kx][ky]; only shapes the synthetic spectrum."""
    kx = cfg.dkx * kx_integers(cfg.Nx)[None, :, None]
    ky = cfg.dky * ky_integers(cfg.Ny)[None, None, :]
    sh = cfg.shat
    kp2 = (ky * ky * geo["gds2"][:, None, None]
           + 2.0 * kx * ky * geo["gds21"][:, None, None] / sh
           + kx * kx * geo["gds22"][:, None, None] / (sh * sh))
    return 1.0 / (1.0 + kp2)


def hermitian_fix_ky0(a: np.ndarray) -> None:
    """In place: make the ky=0 column of [..., kx, ky] arrays satisfy f(-kx,0)=conj f(kx,0),
    and zero the (0,0) mode.  (Reality condition.)"""
    nakx = a.shape[-2]
    K = (nakx - 1) // 2
    # compact order: index i in 1..K is +i, index nakx-i is -i
    pos = a[..., 1:K + 1, 0]
    a[..., nakx - 1:K:-1, 0] = np.conj(pos)
    a[..., 0, 0] = 0.0


def make_state(cfg: Config, geo: dict | None = None, planes=None, hermite_block=None) -> np.ndarray:
    """Seeded g of shape cfg.g_shape, complex64 (generated in fp64, rounded once).

    ``planes``: optional iterable of (s, m) pairs; if given only those (s,m) slabs are filled
    (others are zero) -- lets the large configurations be sampled without 2x600 MB of fp64.
    ``hermite_block``: optional (m0, m1): return only the slab g[:, m0:m1] of the SAME global state (the
    counter-based generator makes any slice reproducible) -- one rank's share in the multi-GPU bench.
    """
    geo = geo or geometry_arrays(cfg)
    env = _envelope(cfg, geo)                       # [z][kx][ky]
    Ns, Nm, Nl, Nz, nakx, naky = cfg.g_shape
    m0, m1 = (0, Nm) if hermite_block is None else hermite_block
    if not (0 <= m0 < m1 <= Nm):
        raise ValueError("hermite_block out of range")
    g = np.zeros((Ns, m1 - m0, Nl, Nz, nakx, naky), dtype=np.complex64)
    per_l = Nz * nakx * naky
    want = None if planes is None else set(planes)
    for s in range(Ns):
        for m in range(m0, m1):
            if want is not None and (s, m) not in want:
                continue
            for l in range(Nl):
                flat0 = ((s * Nm + m) * Nl + l) * per_l      # complex element counter of the global layout
                n = counter_normals(cfg.seed, 2 * flat0, 2 * per_l)
                v = (n[0::2] + 1j * n[1::2]).reshape(Nz, nakx, naky)
                v *= env * (cfg.decay ** (-(l + m))) * cfg.species[s].amp
                hermitian_fix_ky0(v)
                g[s, m - m0, l] = v.astype(np.complex64)
    return g


def random_phi(cfg: Config, geo: dict | None = None, seed_offset: int = 977) -> np.ndarray:
    """A seeded potential with the same envelope (used by tests that want a phi that is
    unrelated to g, e.g. the free-energy invariant which must hold for any phi)."""
    geo = geo or geometry_arrays(cfg)
    env = _envelope(cfg, geo)
    Nz, nakx, naky = cfg.phi_shape
    n = counter_normals(cfg.seed + seed_offset, 0, 2 * Nz * nakx * naky)
    v = (n[0::2] + 1j * n[1::2]).reshape(Nz, nakx, naky) * env
    hermitian_fix_ky0(v)
    return v.astype(np.complex64)
