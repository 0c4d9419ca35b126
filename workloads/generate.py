"""Seeded input DATA for the H.psi workloads (numpy only; no operator arithmetic lives here).

rng(stream) = numpy.random.default_rng(SeedSequence([seed, cfg_id, stream])); streams: 0 atoms,
1 V noise, 2 + 10*ik band coefficients of k-point ik, 3 D.  See DESIGN.md section 4 for the recipe
and for which choices are readings of BASELINE.json where it is silent.
"""
import numpy as np

from .configs import get_config


def _rng(seed, cfg_id, stream):
    return np.random.default_rng(np.random.SeedSequence([int(seed), int(cfg_id), int(stream)]))


def lattice(cfg_id):
    """R (3x3, COLUMNS are lattice vectors, bohr), k-points (reduced), Ecut (Ha), S (FFT box)."""
    cfg = get_config(cfg_id)
    R = np.diag(np.asarray(cfg["cell"], dtype=np.float64))
    kpts = [np.asarray(k, dtype=np.float64) for k in cfg["kpoints"]]
    return R, kpts, float(cfg["Ecut"]), tuple(int(s) for s in cfg["S"])


def atoms_fractional(cfg_id, seed=0):
    """Fractional atom positions [natoms, 3] (they carry both the V Gaussians and the projectors)."""
    cfg = get_config(cfg_id)
    rng = _rng(seed, cfg_id, 0)
    cell = np.asarray(cfg["cell"], dtype=np.float64)
    na = cfg["natoms"]
    rule = cfg["atoms"]
    if rule == "uniform":
        x = rng.random((na, 3))
    elif rule == "clustered":  # Cartesian centre + N(0, (3 bohr)^2) per axis (scaled with the cell for tests)
        sigma = 3.0 * min(1.0, cell.min() / 30.0)
        x = (0.5 * cell + sigma * rng.standard_normal((na, 3))) / cell
    elif rule == "slab":  # uniform in x, y; z in the middle third of the cell
        x = rng.random((na, 3))
        x[:, 2] = (1.0 + x[:, 2]) / 3.0
    elif rule == "lattice6":  # simple-cubic sites + N(0, (0.2 bohr)^2) jitter
        n1 = int(np.ceil(na ** (1.0 / 3.0) - 1e-9))
        g = np.stack(np.meshgrid(np.arange(n1), np.arange(n1), np.arange(n1), indexing="ij"), -1).reshape(-1, 3)
        x = g[:na] / float(n1) + 0.2 * rng.standard_normal((na, 3)) / cell
    else:
        raise ValueError(rule)
    return x - np.floor(x)


def make_vloc(cfg_id, atoms, seed=0):
    """V_loc[j] = (Omega/N) V(r_j), float64 [S0, S1, S2]: periodic Gaussians (depth -2 Ha, width 1 bohr,
    minimum image) on the atoms, plus the config's extra term.  Orthorhombic cells => separable sum."""
    cfg = get_config(cfg_id)
    cell = np.asarray(cfg["cell"], dtype=np.float64)
    S = cfg["S"]
    depth, width = -2.0, 1.0
    fac = []
    for d in range(3):
        r = cell[d] * np.arange(S[d]) / S[d]
        dist = r[None, :] - cell[d] * atoms[:, d][:, None]
        dist -= cell[d] * np.round(dist / cell[d])
        fac.append(np.exp(-dist * dist / (2.0 * width * width)))
    V = depth * np.einsum("ai,aj,ak->ijk", fac[0], fac[1], fac[2], optimize=True)
    extra = cfg["extra"]
    if extra == "noise":
        V = V + 0.01 * _rng(seed, cfg_id, 1).standard_normal(V.shape)
    elif extra == "cavity":
        from scipy.special import erfc
        ax = [cell[d] * np.arange(S[d]) / S[d] - 0.5 * cell[d] for d in range(3)]
        rr = np.sqrt(ax[0][:, None, None] ** 2 + ax[1][None, :, None] ** 2 + ax[2][None, None, :] ** 2)
        radius = 8.0 * min(1.0, cell.min() / 30.0)
        V = V + 0.5 * 0.5 * erfc((radius - rr) / 1.0)
    elif extra == "ramp":
        z = cell[2] * np.arange(S[2]) / S[2]
        V = V + 0.01 * (z - 0.5 * cell[2])[None, None, :]
    volume = float(np.prod(cell))
    N = int(S[0]) * int(S[1]) * int(S[2])
    return np.ascontiguousarray(V * (volume / N))


def make_bands(cfg_id, nG, ik=0, nb=None, seed=0, orthonormalise=True):
    """C complex128 [nb, nG]: i.i.d. N(0,1) + i N(0,1); thin QR; scaled so that C^+ (Omega) C = 1."""
    cfg = get_config(cfg_id)
    nb = int(cfg["nb"] if nb is None else nb)
    rng = _rng(seed, cfg_id, 2 + 10 * ik)
    A = rng.standard_normal((nG, nb)) + 1j * rng.standard_normal((nG, nb))
    volume = float(np.prod(cfg["cell"]))
    if orthonormalise:
        A, _ = np.linalg.qr(A)
        A = A / np.sqrt(volume)
    else:
        A = A / np.sqrt(2.0 * nG * volume)
    return np.ascontiguousarray(A.T)


def make_projectors(cfg_id, iG, k, atoms):
    """P complex128 [np, nG], row j = a * n_lm + lm:
    4 pi (-i)^l |q|^l Y_lm(q^) exp(-|q|^2/2) exp(-2 pi i (iG + k) . x_a),  q = G^T (iG + k),
    written with regular solid harmonics (order: s; py, pz, px; dxy, dyz, dz2, dxz, dx2-y2)."""
    cfg = get_config(cfg_id)
    n_lm = cfg["n_lm"]
    cell = np.asarray(cfg["cell"], dtype=np.float64)
    mk = np.asarray(iG, dtype=np.float64) + np.asarray(k, dtype=np.float64)[None, :]
    q = mk * (2.0 * np.pi / cell)[None, :]
    qx, qy, qz = q[:, 0], q[:, 1], q[:, 2]
    q2 = qx * qx + qy * qy + qz * qz
    radial = np.exp(-0.5 * q2)
    pi = np.pi
    ang = [np.full_like(q2, 1.0 / np.sqrt(4 * pi)),
           np.sqrt(3 / (4 * pi)) * qy, np.sqrt(3 / (4 * pi)) * qz, np.sqrt(3 / (4 * pi)) * qx]
    ls = [0, 1, 1, 1]
    if n_lm == 9:
        ang += [np.sqrt(15 / (4 * pi)) * qx * qy, np.sqrt(15 / (4 * pi)) * qy * qz,
                np.sqrt(5 / (16 * pi)) * (3 * qz * qz - q2), np.sqrt(15 / (4 * pi)) * qx * qz,
                np.sqrt(15 / (16 * pi)) * (qx * qx - qy * qy)]
        ls += [2] * 5
    na = atoms.shape[0]
    P = np.empty((na * n_lm, mk.shape[0]), dtype=np.complex128)
    for a in range(na):
        sf = np.exp(-2j * np.pi * (mk @ atoms[a]))
        for lm in range(n_lm):
            P[a * n_lm + lm] = (4 * pi) * ((-1j) ** ls[lm]) * ang[lm] * radial * sf
    return P


def make_D(cfg_id, seed=0):
    """Real diagonal D, uniform[-1, 1] Ha, one per projector."""
    cfg = get_config(cfg_id)
    return _rng(seed, cfg_id, 3).uniform(-1.0, 1.0, cfg["natoms"] * cfg["n_lm"])


def make_inputs(cfg_id, iG, ik=0, nb=None, seed=0, orthonormalise=True):
    """All inputs of one (config, k-point): dict(C, Vloc, P, D, atoms)."""
    R, kpts, _, _ = lattice(cfg_id)
    atoms = atoms_fractional(cfg_id, seed)
    return dict(atoms=atoms,
                Vloc=make_vloc(cfg_id, atoms, seed),
                C=make_bands(cfg_id, len(iG), ik, nb, seed, orthonormalise),
                P=make_projectors(cfg_id, iG, kpts[ik], atoms),
                D=make_D(cfg_id, seed))
