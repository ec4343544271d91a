"""Seeded generators: models, orientation grids, CTF grids, and the assembled workload dict.
Recipe: SURVEY.md section 8(d) / DESIGN.md section 4.  numpy.random.default_rng([seed, stream])."""
from __future__ import annotations

import math

import numpy as np

from .configs import WorkloadSpec, get_spec
from . import simulate

_STREAM = {"atoms": 1, "grid": 2, "images": 3, "ensemble": 4, "density": 5}


def _rng(spec: WorkloadSpec, stream: str):
    return np.random.default_rng([spec.seed, _STREAM[stream]])


# ----------------------------------------------------------------------------- models
def _ball_points(rng, n, radius):
    pts = np.empty((0, 3))
    while len(pts) < n:
        c = rng.uniform(-radius, radius, size=(2 * n + 16, 3))
        pts = np.concatenate([pts, c[(c ** 2).sum(1) <= radius ** 2]])
    return pts[:n].copy()


def make_atom_model(spec: WorkloadSpec):
    """Uniform-density spheres, centres uniform in a ball (BASELINE.json configs 0-2)."""
    rng = _rng(spec, "atoms")
    xyz = _ball_points(rng, spec.n_atoms, spec.ball_A)
    radius = rng.uniform(spec.radius_A[0], spec.radius_A[1], spec.n_atoms) if spec.radius_A[0] != spec.radius_A[1] \
        else np.full(spec.n_atoms, spec.radius_A[0])
    weight = rng.uniform(spec.weight[0], spec.weight[1], spec.n_atoms) if spec.weight[0] != spec.weight[1] \
        else np.full(spec.n_atoms, spec.weight[0])
    return dict(kind="atoms", xyz=xyz, radius=radius, weight=weight, Kq=4)


def _axis_angle_matrix(axis, ang):
    axis = axis / np.linalg.norm(axis)
    K = np.array([[0, -axis[2], axis[1]], [axis[2], 0, -axis[0]], [-axis[1], axis[0], 0]])
    return np.eye(3) + math.sin(ang) * K + (1 - math.cos(ang)) * (K @ K)


def make_ensemble_models(spec: WorkloadSpec):
    """64 rigid-body hinge perturbations (0-30 deg) of one base structure (BASELINE.json config 4):
    atoms on one side of a seeded plane through the centroid are rotated about a seeded axis through it."""
    base = make_atom_model(spec)
    rng = _rng(spec, "ensemble")
    cen = base["xyz"].mean(0)
    models = []
    for _ in range(spec.n_models):
        normal = rng.normal(size=3)
        normal /= np.linalg.norm(normal)
        axis = rng.normal(size=3)
        ang = math.radians(rng.uniform(0.0, 30.0))
        Rm = _axis_angle_matrix(axis, ang)
        xyz = base["xyz"].copy()
        side = (xyz - cen) @ normal > 0
        xyz[side] = (xyz[side] - cen) @ Rm.T + cen
        models.append(dict(kind="atoms", xyz=xyz, radius=base["radius"].copy(), weight=base["weight"].copy(), Kq=4))
    return models


def make_density_model(spec: WorkloadSpec):
    """128^3 float32 voxel map: sum of seeded isotropic Gaussian blobs (sigma = 2 A), unit amplitude,
    centres uniform in a ball; map origin at voxel n/2 (BASELINE.json config 3)."""
    rng = _rng(spec, "density")
    n, vox = spec.n_vox, spec.pixel_A
    centres = _ball_points(rng, spec.n_blobs, spec.ball_A)
    rho = np.zeros((n, n, n), dtype=np.float64)
    sig = spec.blob_sigma_A
    half = int(math.ceil(5 * sig / vox))
    ax = np.arange(-half, half + 1)
    for c in centres:
        i0 = np.rint(c / vox).astype(int)                      # nearest voxel (x, y, z)
        gx = np.exp(-0.5 * (((i0[0] + ax) * vox - c[0]) / sig) ** 2)
        gy = np.exp(-0.5 * (((i0[1] + ax) * vox - c[1]) / sig) ** 2)
        gz = np.exp(-0.5 * (((i0[2] + ax) * vox - c[2]) / sig) ** 2)
        xs, ys, zs = i0[0] + ax + n // 2, i0[1] + ax + n // 2, i0[2] + ax + n // 2
        okx, oky, okz = (xs >= 0) & (xs < n), (ys >= 0) & (ys < n), (zs >= 0) & (zs < n)
        rho[np.ix_(zs[okz], ys[oky], xs[okx])] += gz[okz][:, None, None] * gy[oky][None, :, None] * gx[okx][None, None, :]
    return dict(kind="density", rho=rho.astype(np.float32), voxel_A=float(vox), blob_centres=centres,
                blob_sigma_A=float(sig))


# ----------------------------------------------------------------------------- orientation grids (R12)
def _qmul(a, b):
    w1, x1, y1, z1 = np.moveaxis(a, -1, 0)
    w2, x2, y2, z2 = np.moveaxis(b, -1, 0)
    return np.stack([w1 * w2 - x1 * x2 - y1 * y2 - z1 * z2, w1 * x2 + x1 * w2 + y1 * z2 - z1 * y2,
                     w1 * y2 - x1 * z2 + y1 * w2 + z1 * x2, w1 * z2 + x1 * y2 - y1 * x2 + z1 * w2], -1)


def euler_zyz_to_quat(alpha, beta, gamma):
    """R = Rz(alpha) Ry(beta) Rz(gamma), active (R12) -> unit quaternion (w, x, y, z)."""
    alpha, beta, gamma = np.broadcast_arrays(np.asarray(alpha, float), np.asarray(beta, float), np.asarray(gamma, float))
    z = np.zeros_like(alpha)
    qa = np.stack([np.cos(alpha / 2), z, z, np.sin(alpha / 2)], -1)
    qb = np.stack([np.cos(beta / 2), z, np.sin(beta / 2), z], -1)
    qg = np.stack([np.cos(gamma / 2), z, z, np.sin(gamma / 2)], -1)
    return _qmul(_qmul(qa, qb), qg)


def euler_grid(na, nb, ng):
    """Uniform in (alpha, cos beta, gamma) at cell mid-points: duplicate-free (no pole, no q == -q)."""
    al = (np.arange(na) + 0.5) * 2 * np.pi / na
    cb = -1 + (np.arange(nb) + 0.5) * 2 / nb
    ga = (np.arange(ng) + 0.5) * 2 * np.pi / ng
    A, B, G = np.meshgrid(al, np.arccos(cb), ga, indexing="ij")
    return euler_zyz_to_quat(A.ravel(), B.ravel(), G.ravel())


def hopf_fibonacci_grid(n_dir, n_psi):
    """Hopf coordinates [39]: n_dir Fibonacci-lattice directions on S2 x n_psi mid-point in-plane angles.
    Stand-in for the HEALPix-based grid of Yershova et al. (not available offline); duplicate-free."""
    i = np.arange(n_dir) + 0.5
    theta = np.arccos(1 - 2 * i / n_dir)
    phi = (np.pi * (1 + 5 ** 0.5) * i) % (2 * np.pi)
    psi = (np.arange(n_psi) + 0.5) * 2 * np.pi / n_psi
    TH, PS = np.meshgrid(theta, psi, indexing="ij")
    PH, _ = np.meshgrid(phi, psi, indexing="ij")
    return euler_zyz_to_quat(PH.ravel(), TH.ravel(), PS.ravel())


def orientation_grid(spec: WorkloadSpec):
    q = euler_grid(*spec.orient_shape) if spec.orient_grid == "euler" else hopf_fibonacci_grid(*spec.orient_shape)
    return np.ascontiguousarray(q[:: spec.orient_stride])


# ----------------------------------------------------------------------------- CTF grid (R8, R9)
def electron_wavelength_A(kV: float) -> float:
    V = kV * 1e3
    return 12.2643 / math.sqrt(V + 0.97845e-6 * V * V)


def ctf_from_defocus(defocus_um: float, bfactor_A2: float, kV: float = 300.0):
    """(a, b) of CTF(s|a,A) Env(s|b) with s = 2 pi k:  a s^2/2 = pi lambda dz k^2  ->  a = lambda dz / (2 pi)  (R8);
    Env = exp(-B k^2/4) -> b = B / (8 pi^2)  (R9)."""
    a = electron_wavelength_A(kV) * defocus_um * 1e4 / (2 * math.pi)
    b = bfactor_A2 / (8 * math.pi ** 2)
    return a, b


def ctf_grid(spec: WorkloadSpec):
    """[C][3] rows (a, A, b); order: defocus slowest, then B-factor, then amplitude contrast."""
    rows = []
    for dz in spec.defocus_um:
        for B in spec.bfactor_A2:
            for A in spec.amp_contrast:
                a, b = ctf_from_defocus(dz, B, spec.kV)
                rows.append((a, A, b))
    return np.array(rows, dtype=np.float64)


# ----------------------------------------------------------------------------- the workload
def build_workload(name_or_spec, with_images: bool = True, **overrides):
    """Returns a dict: spec, models (list), quats [O][4], ctfs [C][3], images float32 [I][N][N], truth (dict of
    planted model / orientation / ctf / dx / dy / N / mu / snr per image)."""
    spec = name_or_spec if isinstance(name_or_spec, WorkloadSpec) else get_spec(name_or_spec, **overrides)
    if spec.model == "atoms":
        models = [make_atom_model(spec)]
    elif spec.model == "ensemble":
        models = make_ensemble_models(spec)
    else:
        models = [make_density_model(spec)]
    quats = orientation_grid(spec)
    ctfs = ctf_grid(spec)
    # The C ABI takes float32 models / grids: round here, once, so that every consumer sees identical numbers.
    r32 = lambda a: np.ascontiguousarray(a, dtype=np.float32).astype(np.float64)
    for m in models:
        if m["kind"] == "atoms":
            m["xyz"], m["radius"], m["weight"] = r32(m["xyz"]), r32(m["radius"]), r32(m["weight"])
    quats, ctfs = r32(quats), r32(ctfs)
    wl = dict(spec=spec, models=models, quats=quats, ctfs=ctfs)
    if with_images:
        rng = _rng(spec, "images")
        I, D = spec.n_images, spec.max_shift
        src_models = np.arange(min(spec.n_source_models, len(models)))
        truth = dict(
            model=src_models[np.arange(I) * len(src_models) // I],      # equal blocks (128 each for Ensemble)
            orient=rng.integers(0, len(quats), I), ctf=rng.integers(0, len(ctfs), I),
            dx=rng.integers(-D, D + 1, I), dy=rng.integers(-D, D + 1, I),
            N=rng.uniform(0.5, 2.0, I), mu_frac=rng.uniform(-1.0, 1.0, I),
            snr=rng.uniform(spec.snr[0], spec.snr[1], I) if spec.snr[0] != spec.snr[1] else np.full(I, spec.snr[0]),
            noise_seed=rng.integers(0, 2 ** 31 - 1, I))
        wl["truth"] = truth
        wl["images"] = simulate.render_images(spec, models, quats, ctfs, truth)
    return wl
