"""FP64 CPU oracle for the BioEM hot path -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Thin ctypes marshalling around ``bioem_oracle.c`` (which holds all of the arithmetic and cites the
paper passage by passage).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package; the product package
``paper_1609_06634_b200`` never does, and this package never imports it.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "bioem_oracle.c"
_LIB = _HERE / "libbioem_oracle.so"

_dp = C.POINTER(C.c_double)
_fp = C.POINTER(C.c_float)
_llp = C.POINTER(C.c_longlong)


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (plain C, OpenMP over images)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        subprocess.check_call(
            ["gcc", "-O3", "-mavx2", "-mfma", "-fopenmp", "-shared", "-fPIC", "-o", str(tmp), str(_SRC), "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(str(_LIB))
        _lib.bo_ctf_env.restype = C.c_double
        _lib.bo_ctf_env.argtypes = [C.c_double] * 4
        _lib.bo_log_post_c1.restype = C.c_double
        _lib.bo_log_post_c1.argtypes = [C.c_double] * 6
        _lib.bo_log_post_c2.restype = C.c_double
        _lib.bo_log_post_c2.argtypes = [C.c_double] * 6
        _lib.bo_const_n.restype = C.c_double
        _lib.bo_const_n.argtypes = [C.c_double]
        _lib.bo_log_lik_eq8.restype = C.c_double
        _lib.bo_log_lik_eq8.argtypes = [C.c_int, _dp, _dp, C.c_double, C.c_double, C.c_double]
        _lib.bo_num_threads.restype = C.c_int
    return _lib


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_dp)


def num_threads() -> int:
    return int(lib().bo_num_threads())


def quat_to_matrix(q):
    q, qp = _d(q)
    R = np.empty(9)
    lib().bo_quat_to_matrix(qp, R.ctypes.data_as(_dp))
    return R.reshape(3, 3)


def project_atoms(xyz, radius, weight, q, N, px, Kq=4):
    """Eq. 1, R10-R12.  Returns I0 [N][N] float64."""
    xyz, xp = _d(xyz)
    radius, rp = _d(radius)
    weight, wp = _d(weight)
    q, qp = _d(q)
    out = np.empty((N, N))
    lib().bo_project_atoms(C.c_int(len(radius)), xp, rp, wp, qp, C.c_int(N), C.c_double(px), C.c_int(Kq),
                           out.ctypes.data_as(_dp))
    return out


def dft2(x, sign=-1, scale=1.0):
    """Eq. 2 (sign=-1) / Eq. 3 (sign=+1, scale=1/N^2), naive separable sums."""
    x = np.asarray(x)
    N = x.shape[0]
    re, rp = _d(x.real)
    im, ip = _d(x.imag) if np.iscomplexobj(x) else (None, None)
    o_re, o_im = np.empty((N, N)), np.empty((N, N))
    lib().bo_dft2(C.c_int(N), rp, ip, C.c_int(sign), C.c_double(scale), o_re.ctypes.data_as(_dp),
                  o_im.ctypes.data_as(_dp))
    return o_re + 1j * o_im


def ctf_env(s2, a, A, b):
    return float(lib().bo_ctf_env(s2, a, A, b))


def apply_ctf(I0, px, a, A, b):
    """Eqs. 2-5: I1 = F^-1(F(I0) CTF Env)."""
    I0, p = _d(I0)
    N = I0.shape[0]
    out = np.empty((N, N))
    lib().bo_apply_ctf(C.c_int(N), C.c_double(px), p, C.c_double(a), C.c_double(A), C.c_double(b),
                       out.ctypes.data_as(_dp))
    return out


def apply_ctf_spectrum(F, px, a, A, b):
    F = np.asarray(F)
    N = F.shape[0]
    re, rp = _d(F.real)
    im, ip = _d(F.imag)
    out = np.empty((N, N))
    lib().bo_apply_ctf_spectrum(C.c_int(N), C.c_double(px), rp, ip, C.c_double(a), C.c_double(A), C.c_double(b),
                                out.ctypes.data_as(_dp))
    return out


def apply_psf_realspace(I0, px, a, A, b):
    """Eq. 6 (tiny images only; a pin for Eq. 5 == Eq. 6)."""
    I0, p = _d(I0)
    N = I0.shape[0]
    out = np.empty((N, N))
    lib().bo_apply_psf_realspace(C.c_int(N), C.c_double(px), p, C.c_double(a), C.c_double(A), C.c_double(b),
                                 out.ctypes.data_as(_dp))
    return out


def _cc(fn, Iobs, I1, D):
    Iobs, ap = _d(Iobs)
    I1, bp = _d(I1)
    N = Iobs.shape[0]
    out = np.empty((2 * D + 1, 2 * D + 1))
    fn(C.c_int(N), ap, bp, C.c_int(D), out.ctypes.data_as(_dp))
    return out


def cross_corr_direct(Iobs, I1, D):
    """C_co[dy+D, dx+D] by direct circular summation (Eq. 7 semantics; the definition)."""
    return _cc(lib().bo_cross_corr_direct, Iobs, I1, D)


def cross_corr_eq12(Iobs, I1, D):
    """Eq. 12 evaluated as a naive double sum (tiny images)."""
    return _cc(lib().bo_cross_corr_eq12, Iobs, I1, D)


def cross_corr_dft(Iobs, I1, D):
    """Tier B: FP64 output-pruned separable DFT (validated against the direct sum, not the definition)."""
    return _cc(lib().bo_cross_corr_dft, Iobs, I1, D)


def log_post_c1(n, Co, Coo, Cc, Ccc, Cco):
    return float(lib().bo_log_post_c1(n, Co, Coo, Cc, Ccc, Cco))


def log_post_c2(n, Co, Coo, Cc, Ccc, Cco):
    return float(lib().bo_log_post_c2(n, Co, Coo, Cc, Ccc, Cco))


def const_n(n):
    return float(lib().bo_const_n(float(n)))


def log_lik_eq8(Iobs, I1s, N_, mu, lam):
    Iobs, ap = _d(np.ravel(Iobs))
    I1s, bp = _d(np.ravel(I1s))
    return float(lib().bo_log_lik_eq8(C.c_int(Iobs.size), ap, bp, N_, mu, lam))


def dft3(rho):
    rho, p = _d(rho)
    N = rho.shape[0]
    vr, vi = np.empty((N, N, N)), np.empty((N, N, N))
    lib().bo_dft3(C.c_int(N), p, vr.ctypes.data_as(_dp), vi.ctypes.data_as(_dp))
    return vr + 1j * vi


def fourier_slice(V, voxel_A, q):
    """R21: central section of the 3-D DFT V [kz][ky][kx] -> full 2-D spectrum [m][l]."""
    V = np.asarray(V)
    N = V.shape[0]
    vr, rp = _d(V.real)
    vi, ip = _d(V.imag)
    q, qp = _d(q)
    fr, fi = np.empty((N, N)), np.empty((N, N))
    lib().bo_fourier_slice(C.c_int(N), rp, ip, C.c_double(voxel_A), qp, fr.ctypes.data_as(_dp),
                           fi.ctypes.data_as(_dp))
    return fr + 1j * fi


def calc_image(model, q, ctf, N, px):
    """I1 for one (model, orientation, CTF) -- Eqs. 1-5.  model: dict(kind='atoms', xyz, radius, weight)
    or dict(kind='density', V=<3-D DFT>, voxel_A)."""
    a, A, b = ctf
    if model["kind"] == "atoms":
        I0 = project_atoms(model["xyz"], model["radius"], model["weight"], q, N, px, model.get("Kq", 4))
        return apply_ctf(I0, px, a, A, b)
    F = fourier_slice(model["V"], model["voxel_A"], q)
    return apply_ctf_spectrum(F, px, a, A, b)


def prepare_model(model):
    """Density models: attach the 3-D DFT (computed once)."""
    if model["kind"] == "density" and "V" not in model:
        model = dict(model)
        model["V"] = dft3(model["rho"])
    return model


class RunState:
    """Running accumulators of Eq. 9 for one model: log-sum-exp (m, s), best, second best, argmax."""

    def __init__(self, n_img):
        self.m = np.full(n_img, -np.inf)
        self.s = np.zeros(n_img)
        self.best = np.full(n_img, -np.inf)
        self.second = np.full(n_img, -np.inf)
        self.best_flat = np.full(n_img, -1, dtype=np.int64)

    def log_posterior(self):
        return self.m + np.log(self.s)


def cropped_sums(obs, I1, D):
    """Real-space cropping variant (R25): (C_co(d), C_c(d), C_cc(d)), each [2D+1][2D+1] indexed [dy+D][dx+D]."""
    obs, op = _d(obs)
    I1, ip = _d(I1)
    N, S1 = obs.shape[0], 2 * D + 1
    out = [np.empty((S1, S1)) for _ in range(3)]
    lib().bo_cropped_sums(C.c_int(N), op, ip, C.c_int(D), *[o.ctypes.data_as(_dp) for o in out])
    return tuple(out)


def run_model(model, N, px, D, quats, ctfs, images, lp_orient=None, lp_ctf=None, o_begin=0, o_end=None,
              tier=0, state=None):
    """Eq. 9 on the grid for ONE model: all orientations in [o_begin, o_end) x CTFs x shifts, every image.
    ctfs: array [C][3] of (a, A, b).  images: float32 [I][N][N].  Returns RunState (chunks may be chained)."""
    model = prepare_model(model)
    quats, qp = _d(quats)
    ctfs = np.ascontiguousarray(ctfs, dtype=np.float64)
    ca, cap = _d(ctfs[:, 0])
    cA, cAp = _d(ctfs[:, 1])
    cb, cbp = _d(ctfs[:, 2])
    images = np.ascontiguousarray(images, dtype=np.float32)
    n_img = images.shape[0]
    st = state or RunState(n_img)
    o_end = len(quats) if o_end is None else o_end
    lpo = lpo_p = lpc = lpc_p = None
    if lp_orient is not None:
        lpo, lpo_p = _d(lp_orient)
    if lp_ctf is not None:
        lpc, lpc_p = _d(lp_ctf)
    null = C.cast(None, _dp)
    if model["kind"] == "atoms":
        xyz, xp = _d(model["xyz"])
        rad, rp = _d(model["radius"])
        wt, wp = _d(model["weight"])
        kind, nat, Kq = 0, len(rad), int(model.get("Kq", 4))
        vr_p = vi_p = null
        vox = 0.0
    else:
        V = model["V"]
        vr, vr_p = _d(V.real)
        vi, vi_p = _d(V.imag)
        kind, nat, Kq = 1, 0, 0
        xp = rp = wp = null
        vox = float(model["voxel_A"])
    rc = lib().bo_run(
        C.c_int(N), C.c_double(px), C.c_int(D), C.c_int(kind),
        C.c_int(nat), xp, rp, wp, C.c_int(Kq), vr_p, vi_p, C.c_double(vox),
        C.c_int(len(quats)), qp, lpo_p if lpo is not None else null,
        C.c_int(len(ctfs)), cap, cAp, cbp, lpc_p if lpc is not None else null,
        C.c_int(n_img), images.ctypes.data_as(_fp), C.c_int(o_begin), C.c_int(o_end), C.c_int(tier),
        st.m.ctypes.data_as(_dp), st.s.ctypes.data_as(_dp), st.best.ctypes.data_as(_dp),
        st.second.ctypes.data_as(_dp), st.best_flat.ctypes.data_as(_llp))
    assert rc == 0
    return st


def orientation_log_posterior(model, N, px, D, quats, ctfs, images, lp_orient=None, lp_ctf=None):
    """Posterior as a function of the orientation (the paper's third output): for every image and orientation o,
    log sum_{ctf, d} w(o, ctf, d) P(o, ctf, d) -- Eq. 9's sum restricted to one orientation, weights of the FULL grid, so that
    the log-sum-exp over o is log_posterior.  Returns [I][O].  Plain restatement: one run of the loop nest per orientation."""
    out = np.empty((np.asarray(images).shape[0], len(quats)))
    for o in range(len(quats)):
        out[:, o] = run_model(model, N, px, D, quats, ctfs, images, lp_orient, lp_ctf, o_begin=o, o_end=o + 1).log_posterior()
    return out


def ensemble_log_posterior(logp, weights=None):
    """Eq. 10: log P(M|Omega) = sum_omega log sum_m w_m P_m,omega up to the constant the paper drops.
    logp: [I][M] log-posteriors; weights: [M] (None = 1/M).  Returns (total, per_image)."""
    logp = np.asarray(logp, dtype=np.float64)
    w = np.full(logp.shape[1], 1.0 / logp.shape[1]) if weights is None else np.asarray(weights, dtype=np.float64)
    per = np.empty(logp.shape[0])
    for i in range(logp.shape[0]):
        with np.errstate(divide="ignore"):
            t = logp[i] + np.log(w)
        m = t.max()
        per[i] = m + math.log(sum(math.exp(x - m) for x in t)) if m > -np.inf else -np.inf
    return float(per.sum()), per


def synthetic_map(I1, dx, dy, obs=None, crop=False):
    """Synthetic map ("print the synthetic map corresponding to a specific parameter set theta") for
    theta = (orientation, CTF parameters: the calculated image I1 of Eqs. 1-5; centre displacement d = (dx, dy);
    normalisation N and offset mu), which is I_cal of Eq. 7:   S(k, j) = N * I_d(k, j) - mu,   with the displaced image of
    bo_cross_corr_direct / bo_cropped_sums: I_d(k, j) = I1((k + dy) mod n, (j + dx) mod n) (Fourier variant, R5), or, with
    crop=True (real-space variant, R25), I1(k + dy, j + dx) inside the box and 0 outside.
    obs=None: N = 1, mu = 0.  Otherwise (N, mu) are the values that maximise the likelihood of Eq. 8 for that image at any
    lambda, i.e. that minimise sum (obs - N I_d + mu)^2; setting both derivatives to zero (the sums in the paper's notation):
        N = (n C_co - C_o C_c) / (n C_cc - C_c^2),      mu = (N C_c - C_o) / n       (Eq. 7 SUBTRACTS mu).
    Returns (S, N, mu).  Plain loops over the pixels."""
    I1 = np.asarray(I1, dtype=np.float64)
    n1 = I1.shape[0]
    Id = np.zeros_like(I1)
    for k in range(n1):
        for j in range(n1):
            k2, j2 = k + dy, j + dx
            if crop:
                if 0 <= k2 < n1 and 0 <= j2 < n1:
                    Id[k, j] = I1[k2, j2]
            else:
                Id[k, j] = I1[k2 % n1, j2 % n1]
    if obs is None:
        return Id, 1.0, 0.0
    obs = np.asarray(obs, dtype=np.float64)
    n = float(n1 * n1)
    Co = Cc = Ccc = Cco = 0.0
    for k in range(n1):
        for j in range(n1):
            Co += obs[k, j]; Cc += Id[k, j]; Ccc += Id[k, j] * Id[k, j]; Cco += obs[k, j] * Id[k, j]
    N_ = (n * Cco - Co * Cc) / (n * Ccc - Cc * Cc)
    mu = (N_ * Cc - Co) / n
    return N_ * Id - mu, N_, mu


def shift_map(image, I1, D, logw, tier=0):
    """log P(C1) + logw for every shift of one (image, calc image) pair: [dy+D][dx+D]."""
    image = np.ascontiguousarray(image, dtype=np.float32)
    I1, ip = _d(I1)
    N = image.shape[0]
    out = np.empty((2 * D + 1, 2 * D + 1))
    lib().bo_shift_map(C.c_int(N), C.c_int(D), image.ctypes.data_as(_fp), ip, C.c_double(logw), C.c_int(tier),
                       out.ctypes.data_as(_dp))
    return out


def unflatten(flat, n_ctf, D):
    """flat index -> (orientation, ctf, dx, dy)  (R15)."""
    S1 = 2 * D + 1
    flat = np.asarray(flat, dtype=np.int64)
    dx = flat % S1 - D
    dy = (flat // S1) % S1 - D
    oc = flat // (S1 * S1)
    return oc // n_ctf, oc % n_ctf, dx, dy


def uniform_logw(n_orient, n_ctf, D):
    return -math.log(n_orient) - math.log(n_ctf) - math.log((2 * D + 1) ** 2)
