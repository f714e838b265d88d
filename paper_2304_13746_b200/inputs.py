"""Seeded synthetic inputs for the five BASELINE.json configurations (and the paper's own 3D
Orszag-Tang benchmark).

This module holds NO arithmetic of the method (no conversion to conserved variables, no reconstruction,
no solver): it only produces primitive cell fields (rho, vx, vy, vz, p) and a discretely divergence-free
staggered field bface = discrete curl of an edge-sampled vector potential.  The same arrays are handed to
the CPU oracle and to the CUDA library, so generator details cannot affect parity.  It imports neither of
them.  Recipes: SURVEY.md §8(d) / DESIGN.md "Input recipe".

All arrays are float64, layout [var][nz][ny][nx] (x fastest); cell centres at (i+1/2) dx on the unit cube;
bface[d][k][j][i] is B_d on the LEFT d-face of cell (i,j,k).
"""
import math

import numpy as np
import torch

SOLVER_HLL, SOLVER_HLLC, SOLVER_HLLD, SOLVER_ROE, SOLVER_RUSANOV = 0, 1, 2, 3, 4
LIMITER_FLAT, LIMITER_MINMOD, LIMITER_VANLEER, LIMITER_LIMO3 = 0, 1, 2, 3
EMF_NONE, EMF_ARITHMETIC, EMF_UCT_CONTACT, EMF_UCT_0, EMF_UCT_HLL = 0, 1, 2, 3, 4

GAMMA = 5.0 / 3.0

# name -> (N, steps, cfl, solver, limiter, emf, seed)
CONFIGS = {
    "config1": dict(n=32, steps=10, cfl=0.3, solver=SOLVER_HLLD, limiter=LIMITER_VANLEER, emf=EMF_ARITHMETIC, seed=1001),
    "config2": dict(n=128, steps=50, cfl=0.4, solver=SOLVER_HLLC, limiter=LIMITER_MINMOD, emf=EMF_NONE, seed=1002),
    "config3": dict(n=128, steps=50, cfl=0.3, solver=SOLVER_HLLD, limiter=LIMITER_VANLEER, emf=EMF_UCT_CONTACT, seed=1003),
    "config4": dict(n=256, steps=20, cfl=0.3, solver=SOLVER_ROE, limiter=LIMITER_VANLEER, emf=EMF_ARITHMETIC, seed=1004),
    "config5": dict(n=512, steps=20, cfl=0.3, solver=SOLVER_HLLD, limiter=LIMITER_VANLEER, emf=EMF_UCT_CONTACT, seed=1005),
}


def half_space_modes(kmax):
    """Integer wavevectors with 0 < |k| <= kmax, one of each +-k pair, in a fixed (kz, ky, kx) order."""
    out = []
    for kz in range(0, kmax + 1):
        for ky in range(-kmax, kmax + 1):
            for kx in range(-kmax, kmax + 1):
                if kx * kx + ky * ky + kz * kz > kmax * kmax or (kx, ky, kz) == (0, 0, 0):
                    continue
                if kz > 0 or (kz == 0 and ky > 0) or (kz == 0 and ky == 0 and kx > 0):
                    out.append((kx, ky, kz))
    return out


def random_phase_field(n, modes, phases, offset, device="cpu"):
    """sum_k cos(2 pi k.x + phi_k) sampled at x = (index + offset) / n, by one inverse FFT."""
    spec = torch.zeros((n, n, n), dtype=torch.complex128, device=device)
    ox, oy, oz = offset
    for (kx, ky, kz), ph in zip(modes, phases):
        a = ph + 2.0 * math.pi * (kx * ox + ky * oy + kz * oz) / n
        spec[kz % n, ky % n, kx % n] += complex(math.cos(a), math.sin(a))
    f = torch.fft.ifftn(spec).real * float(n) ** 3
    return f.contiguous()


def curl_edges_to_faces(ax, ay, az, dx):
    """Discrete curl.  ax[k,j,i] sits on the x-edge (i, j-1/2, k-1/2), ay on (i-1/2, j, k-1/2), az on
    (i-1/2, j-1/2, k); the result sits on the left faces, periodic."""
    def up(a, dim):
        return torch.roll(a, shifts=-1, dims=dim)
    bx = ((up(az, 1) - az) - (up(ay, 0) - ay)) / dx
    by = ((up(ax, 0) - ax) - (up(az, 2) - az)) / dx
    bz = ((up(ay, 2) - ay) - (up(ax, 1) - ax)) / dx
    return torch.stack([bx, by, bz])


def _centres(n, device):
    x = (torch.arange(n, dtype=torch.float64, device=device) + 0.5) / n
    return x.view(1, 1, n), x.view(1, n, 1), x.view(n, 1, 1)


def _random_velocity(rng, n, kmax, device):
    modes = half_space_modes(kmax)
    v = []
    for _ in range(3):
        ph = rng.uniform(0.0, 2.0 * math.pi, size=len(modes))
        v.append(random_phase_field(n, modes, ph, (0.5, 0.5, 0.5), device))
    return torch.stack(v)


def _random_potential_curl(rng, n, kmax, device):
    modes = half_space_modes(kmax)
    offs = [(0.5, 0.0, 0.0), (0.0, 0.5, 0.0), (0.0, 0.0, 0.5)]
    a = []
    for o in offs:
        ph = rng.uniform(0.0, 2.0 * math.pi, size=len(modes))
        a.append(random_phase_field(n, modes, ph, o, device))
    return curl_edges_to_faces(a[0], a[1], a[2], 1.0 / n)


def _scale_rms(v, target_rms):
    rms = torch.sqrt((v * v).sum(dim=0).mean())
    return v * (target_rms / rms)


def orszag_tang_2d(n, seed, device="cpu"):
    """BASELINE config 1 (2D Orszag-Tang of PAPER.md:282-292 extended in z, plus density noise)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    X, Y, _ = _centres(n, device)
    dx = 1.0 / n
    b0 = 1.0 / math.sqrt(4.0 * math.pi)
    noise = torch.from_numpy(rng.uniform(-1e-3, 1e-3, size=(n, n, n))).to(device)
    prim = torch.empty((5, n, n, n), dtype=torch.float64, device=device)
    prim[0] = 25.0 / (36.0 * math.pi) + noise
    prim[1] = (-torch.sin(2 * math.pi * Y)).expand(n, n, n)
    prim[2] = (torch.sin(2 * math.pi * X)).expand(n, n, n)
    prim[3] = 0.0
    prim[4] = 5.0 / (12.0 * math.pi)
    e = torch.arange(n, dtype=torch.float64, device=device) / n      # edge coordinates i*dx
    az = (b0 / (4 * math.pi)) * torch.cos(4 * math.pi * e).view(1, 1, n) + \
         (b0 / (2 * math.pi)) * torch.cos(2 * math.pi * e).view(1, n, 1)
    az = az.expand(n, n, n).contiguous()
    zero = torch.zeros_like(az)
    bface = curl_edges_to_faces(zero, zero, az, dx)
    return prim, bface.contiguous()


def orszag_tang_3d(n, device="cpu"):
    """The paper's performance workload.  Each B component is independent of its own
    coordinate, so point samples at face centres are discretely divergence-free."""
    X, Y, Z = _centres(n, device)
    b0 = 1.0 / math.sqrt(4.0 * math.pi)
    two_pi = 2 * math.pi
    prim = torch.empty((5, n, n, n), dtype=torch.float64, device=device)
    prim[0] = 25.0 / (36.0 * math.pi)
    prim[1] = (-torch.sin(two_pi * Y)).expand(n, n, n)
    prim[2] = (torch.sin(two_pi * X) + torch.cos(two_pi * Z)).expand(n, n, n)
    prim[3] = torch.cos(two_pi * X).expand(n, n, n)
    prim[4] = 5.0 / (12.0 * math.pi)
    bface = torch.empty((3, n, n, n), dtype=torch.float64, device=device)
    bface[0] = (-b0 * torch.sin(two_pi * Y)).expand(n, n, n)
    bface[1] = (b0 * torch.sin(2 * two_pi * X)).expand(n, n, n)
    bface[2] = (b0 * (torch.cos(two_pi * X) + torch.sin(two_pi * Y))).expand(n, n, n)
    return prim, bface


def sedov(n, r_i=None, device="cpu"):
    """The paper's Cartesian Sedov-Taylor blast: rho = 1, P = 1e-2 at rest, gamma = 5/3, and an energy
    E = 1 deposited as pressure in the cells whose centres lie within r_i of the box centre (periodic unit cube; the
    paper does not print r_i: 3.5 cells unless given).  Returns (prim, the deposited energy as discretised = 1)."""
    r_i = 3.5 / n if r_i is None else r_i
    x = (torch.arange(n, dtype=torch.float64, device=device) + 0.5) / n - 0.5
    r2 = x.view(1, 1, n) ** 2 + x.view(1, n, 1) ** 2 + x.view(n, 1, 1) ** 2
    inside = r2 < r_i * r_i
    n_in = int(inside.sum())
    prim = torch.zeros((5, n, n, n), dtype=torch.float64, device=device)
    prim[0] = 1.0
    prim[4] = 1e-2
    prim[4][inside] = (GAMMA - 1.0) * 1.0 / (n_in * (1.0 / n) ** 3)
    return prim, n_in


def turbulence_hd(n, seed, kmax, mach, device="cpu"):
    """BASELINE config 2: rho = p = 1, random-phase velocity with rms Mach `mach`."""
    rng = np.random.Generator(np.random.PCG64(seed))
    v = _scale_rms(_random_velocity(rng, n, kmax, device), mach * math.sqrt(GAMMA))
    prim = torch.empty((5, n, n, n), dtype=torch.float64, device=device)
    prim[0] = 1.0
    prim[1:4] = v
    prim[4] = 1.0
    return prim, None


def turbulence_mhd(n, seed, kmax, mach, beta, device="cpu"):
    """BASELINE configs 3 and 5: rho = p = 1, random-phase v (rms Mach) and B = curl A with plasma beta."""
    rng = np.random.Generator(np.random.PCG64(seed))
    v = _scale_rms(_random_velocity(rng, n, kmax, device), mach * math.sqrt(GAMMA))
    b = _scale_rms(_random_potential_curl(rng, n, kmax, device), math.sqrt(2.0 / beta))
    prim = torch.empty((5, n, n, n), dtype=torch.float64, device=device)
    prim[0] = 1.0
    prim[1:4] = v
    prim[4] = 1.0
    return prim, b.contiguous()


def turbulence_mhd_lognormal(n, seed, kmax, mach, beta, bz0, sigma, device="cpu"):
    """BASELINE config 4: lognormal density, Mach-2 velocity, mean field (0,0,bz0) + curl A, total beta."""
    rng = np.random.Generator(np.random.PCG64(seed))
    v = _scale_rms(_random_velocity(rng, n, kmax, device), mach * math.sqrt(GAMMA))
    b = _random_potential_curl(rng, n, kmax, device)
    gauss = torch.from_numpy(rng.standard_normal(size=(n, n, n))).to(device)
    # <|B0 + s b|^2> = 2 p / beta  =>  s^2 <b^2> + 2 s <B0.b> + (B0^2 - 2/beta) = 0
    qa = float((b * b).sum(dim=0).mean())
    qb = 2.0 * bz0 * float(b[2].mean())
    qc = bz0 * bz0 - 2.0 / beta
    s = (-qb + math.sqrt(qb * qb - 4.0 * qa * qc)) / (2.0 * qa)
    b = b * s
    b[2] += bz0
    prim = torch.empty((5, n, n, n), dtype=torch.float64, device=device)
    prim[0] = torch.exp(sigma * gauss - 0.5 * sigma * sigma)
    prim[1:4] = v
    prim[4] = 1.0
    return prim, b.contiguous()


def make(name, n=None, device="cpu"):
    """Returns (prim, bface_or_None, meta).  `n` overrides the grid size (tests use reduced sizes with the
    same recipe; DESIGN.md says where)."""
    cfg = dict(CONFIGS[name])
    if n is not None:
        cfg["n"] = n
    N, seed = cfg["n"], cfg["seed"]
    if name == "config1":
        prim, b = orszag_tang_2d(N, seed, device)
    elif name == "config2":
        prim, b = turbulence_hd(N, seed, 4, 0.5, device)
    elif name == "config3":
        prim, b = turbulence_mhd(N, seed, 4, 1.0, 10.0, device)
    elif name == "config4":
        prim, b = turbulence_mhd_lognormal(N, seed, 8, 2.0, 1.0, 0.1, 0.1, device)
    elif name == "config5":
        prim, b = turbulence_mhd(N, seed, 8, 1.0, 10.0, device)
    else:
        raise KeyError(name)
    cfg.update(dx=1.0 / N, gamma=GAMMA, name=name)
    return prim.contiguous(), b, cfg
