"""Synthetic microscope: renders the noisy particle images of a workload (input synthesis only).

It stands in for the paper's experimental particle sets (Frh, GroEL), which are not available.
Each image is  N * (projection of a model at a grid orientation, convolved with a grid CTF)  circularly displaced
by an integer (dx, dy), plus an offset mu and i.i.d. Gaussian noise at a given SNR (BASELINE.json configs;
SNR = var(N * signal) / sigma_noise^2, R18).  The renderer is deliberately its OWN code (vectorised numpy + numpy's
FFT): the CUDA library and the CPU oracle never call it and it calls neither, so a mistake here can only make the
inputs less realistic -- it cannot make the two sides agree.  tests/test_workloads.py checks that it renders the
same forward model as the oracle (so planted parameters are the best-scoring ones).
"""
from __future__ import annotations

import math
import os

import numpy as np


def _rot(q):
    w, x, y, z = np.asarray(q, float) / np.linalg.norm(q)
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                     [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                     [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])


def render_atoms(model, q, N, px):
    """Pixel-integrated z-projection of uniform spheres, K x K mid-point sub-sampling per pixel."""
    K = int(model.get("Kq", 4))
    R = _rot(q)
    xy = model["xyz"] @ R[:2].T
    rad, wt = model["radius"], model["weight"]
    dens = wt / (4.0 / 3.0 * math.pi * rad ** 3)
    jc = np.rint(xy[:, 0] / px).astype(np.int64)
    kc = np.rint(xy[:, 1] / px).astype(np.int64)
    hw = int(math.ceil(rad.max() / px)) + 1
    h = px / K
    img = np.zeros(N * N)
    sub = (np.arange(K) + 0.5) * h - 0.5 * px
    for oy in range(-hw, hw + 1):
        for ox in range(-hw, hw + 1):
            j, k = jc + ox, kc + oy
            acc = np.zeros(len(rad))
            for sy in sub:
                dy2 = (k * px + sy - xy[:, 1]) ** 2
                for sx in sub:
                    d2 = rad ** 2 - (j * px + sx - xy[:, 0]) ** 2 - dy2
                    acc += 2.0 * np.sqrt(np.maximum(d2, 0.0))
            jj, kk = j + N // 2, k + N // 2
            ok = (jj >= 0) & (jj < N) & (kk >= 0) & (kk < N) & (acc > 0)
            img += np.bincount(kk[ok] * N + jj[ok], weights=(dens * acc * h * h)[ok], minlength=N * N)
    return img.reshape(N, N)


def ctf_image(N, px, a, A, b):
    """CTF(s)Env(s) on the rfft2 grid [m][l], s = 2 pi (l', m') / (N px)."""
    m = np.fft.fftfreq(N, d=1.0 / N)[:, None]
    l = np.arange(N // 2 + 1)[None, :]
    s2 = (2 * math.pi / (N * px)) ** 2 * (l * l + m * m)
    return (-A * np.cos(0.5 * a * s2) - math.sqrt(1 - A * A) * np.sin(0.5 * a * s2)) * np.exp(-0.5 * b * s2)


def density_spectrum(model):
    """3-D DFT of the voxel map with the origin moved to voxel n/2."""
    rho = np.asarray(model["rho"], dtype=np.float64)
    n = rho.shape[0]
    V = np.fft.fftn(rho)
    k = np.fft.fftfreq(n, d=1.0 / n).astype(np.int64)
    sgn = 1 - 2 * (np.abs(k) % 2)
    return V * sgn[:, None, None] * sgn[None, :, None] * sgn[None, None, :]


def render_density_spectrum(Vc, voxel_A, q, N):
    """Central section by trilinear interpolation, half-plane -> rfft2-layout spectrum [m][l]."""
    R = _rot(q)
    h = N // 2
    ms = np.fft.fftfreq(N, d=1.0 / N)[:, None] * np.ones((1, h + 1))
    ls = np.arange(h + 1)[None, :] * np.ones((N, 1))
    kx = R[0, 0] * ls + R[1, 0] * ms
    ky = R[0, 1] * ls + R[1, 1] * ms
    kz = R[0, 2] * ls + R[1, 2] * ms
    inside = (np.abs(kx) <= h - 1) & (np.abs(ky) <= h - 1) & (np.abs(kz) <= h - 1) & (np.abs(ms) < h) & (ls < h)
    fx, fy, fz = np.floor(kx), np.floor(ky), np.floor(kz)
    tx, ty, tz = kx - fx, ky - fy, kz - fz
    out = np.zeros((N, h + 1), dtype=np.complex128)
    for cz in (0, 1):
        for cy in (0, 1):
            for cx in (0, 1):
                w = (tx if cx else 1 - tx) * (ty if cy else 1 - ty) * (tz if cz else 1 - tz)
                ix = (fx + cx).astype(np.int64) % N
                iy = (fy + cy).astype(np.int64) % N
                iz = (fz + cz).astype(np.int64) % N
                out += w * Vc[iz, iy, ix]
    sg = 1 - 2 * ((np.abs(ls) + np.abs(ms)).astype(np.int64) % 2)
    out = np.where(inside, out * sg * voxel_A, 0.0)
    # exact Hermitian symmetry of the self-conjugate column l = 0 (taken from m' >= 0)
    out[h + 1:, 0] = np.conj(out[1:h, 0][::-1])
    out[0, 0] = out[0, 0].real
    return out


def render_signal(model, q, ctf, N, px, cache=None):
    a, A, b = ctf
    if model["kind"] == "atoms":
        spec0 = np.fft.rfft2(render_atoms(model, q, N, px))
    else:
        if cache is not None and "Vc" in cache:
            Vc = cache["Vc"]
        else:
            Vc = density_spectrum(model)
            if cache is not None:
                cache["Vc"] = Vc
        spec0 = render_density_spectrum(Vc, model["voxel_A"], q, N)
    return np.fft.irfft2(spec0 * ctf_image(N, px, a, A, b), s=(N, N))


def _render_block(args):
    spec, models, quats, ctfs, truth, lo, hi = args
    N, px = spec.n_pix, spec.pixel_A
    out = np.empty((hi - lo, N, N), dtype=np.float32)
    caches = [dict() for _ in models]
    for i in range(lo, hi):
        mi = int(truth["model"][i])
        sig = render_signal(models[mi], quats[truth["orient"][i]], ctfs[truth["ctf"][i]], N, px, caches[mi])
        # I_obs(r) = N * I1(r + d) + mu + noise  (Eq. 7 with reading R4), circular (R5)
        sig = truth["N"][i] * np.roll(sig, shift=(-int(truth["dy"][i]), -int(truth["dx"][i])), axis=(0, 1))
        sd = sig.std()
        noise = np.random.default_rng(int(truth["noise_seed"][i])).normal(size=(N, N))
        out[i - lo] = (sig + truth["mu_frac"][i] * sd + noise * sd / math.sqrt(truth["snr"][i])).astype(np.float32)
    return out


def render_images(spec, models, quats, ctfs, truth, workers=None):
    """Every image is rendered from its own parameters and its own noise seed, so the stack can be rendered in blocks by
    worker processes (spawned, not forked: the caller may hold a CUDA context) with a result identical to the serial loop."""
    I = len(truth["orient"])
    if workers is None:
        workers = min(os.cpu_count() or 1, 32, I // 32)
    if workers <= 1:
        return _render_block((spec, models, quats, ctfs, truth, 0, I))
    import multiprocessing as mp
    from concurrent.futures import ProcessPoolExecutor
    # only the models that generate images travel to the workers (a density map is 8 MB, an atom model a few hundred KB)
    used = sorted(set(int(m) for m in truth["model"]))
    slim = [models[m] if m in used else None for m in range(len(models))]
    edges = np.linspace(0, I, 4 * workers + 1).astype(int)
    jobs = [(spec, slim, quats, ctfs, truth, int(a), int(b)) for a, b in zip(edges[:-1], edges[1:]) if b > a]
    with ProcessPoolExecutor(max_workers=workers, mp_context=mp.get_context("spawn")) as ex:
        return np.concatenate(list(ex.map(_render_block, jobs)), axis=0)
