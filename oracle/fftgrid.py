"""Tier C of the CPU oracle -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

The same Eq. 9 grid sum as ``bioem_oracle.c:bo_run`` (tier A, the definition: direct circular summation), with the three
O(N^3) / O(N^2 S) steps replaced by numpy's FFT, a library primitive: the 2-D DFT of the projection (Eq. 2), the
inverse DFT after the CTF multiply (Eqs. 3-5) and the cross term C_co(d) for all displacements from one inverse
transform of conj(I_obs^) I1^ (Eqs. 11-12; reading R3/R4: ``irfft2(conj(O) * I1)[dy mod N, dx mod N]``).
Everything else follows tier A line by line in FP64 / long double: the projection (``bo_project_atoms`` / ``bo_fourier_slice``
of the C file are called as they stand), the sums C_o, C_oo, C_c, C_cc over pixels ("Eqs. S3-S6"), the closed form (C1)
(long double as in ``bo_log_post_c1``), the weights (R7), the log-sum-exp in loop order (R16) and the
strict-greater argmax (R15).

Why it exists: the full grid of a BASELINE.json-sized config is 1e8-5e8 terms per image, and tier A needs n = N^2 multiply-adds
per term plus two naive O(N^3) transforms per calculated image -- hours for the 224^2 config.  Tier C does an image's full grid
in about a minute per core, so the CUDA path's log-posteriors can be compared with an oracle value on the FULL grid, in the
launch configuration bench.py times (SURVEY 8(c) "Parity protocol").

It is NOT the definition.  Pins (tests/test_oracle_pins.py, tests/test_gpu_parity.py): on Tiny and on the mini configs its
log-posteriors, best terms and argmax agree with tier A to 1e-8 / exactly; on every full-size config its shift maps agree
with tier A's direct summation on seeded (image, orientation, CTF) tuples to 1e-7.
"""
from __future__ import annotations

import math
import os

import numpy as np

from . import fourier_slice, prepare_model, project_atoms, RunState, lib  # noqa: F401  (the C steps, as they stand)


def ctf_env_table(N, px, a, A, b):
    """CTF(s|a,A) Env(s|b) (Eqs. 4-5) on the full DFT grid [m][l], |s|^2 from signed frequencies."""
    f = np.fft.fftfreq(N, d=1.0 / N)
    f[N // 2] = N // 2                                       # tier A counts the Nyquist bin as +N/2 (squares: no difference)
    s2 = (2.0 * math.pi / (N * px)) ** 2 * (f[None, :] ** 2 + f[:, None] ** 2)
    ph = 0.5 * a * s2
    return (-A * np.cos(ph) - math.sqrt(1.0 - A * A) * np.sin(ph)) * np.exp(-0.5 * b * s2)


def const_n(n):
    return -0.5 * (n - 2.0) * math.log(2.0 * math.pi) + 0.5 * (n - 5.0) * math.log(2.0) + math.lgamma(0.5 * (n - 3.0))


def log_post_c1(n, Co, Coo, Cc, Ccc, Cco):
    """(C1), vectorised over Cco (and Co, Coo broadcast), in long double like bo_log_post_c1, with its R14 clamp."""
    ld = np.longdouble
    n_, Co, Coo, Cc, Ccc, Cco = ld(n), np.asarray(Co, ld), np.asarray(Coo, ld), ld(Cc), ld(Ccc), np.asarray(Cco, ld)
    Tc = n_ * Ccc - Cc * Cc
    F = n_ * (Coo * Ccc - Cco * Cco) + ld(2) * Co * Cco * Cc - Ccc * Co * Co - Coo * Cc * Cc
    Fmin = ld(1e-300) * Tc * (n_ * Coo - Co * Co) / n_
    F = np.maximum(F, Fmin)
    return (ld(const_n(float(n))) + (n_ / 2 - 2) * np.log(Tc) + (ld(1.5) - n_ / 2) * np.log(F)).astype(np.float64)


def calc_image_fft(model, q, K, N, px):
    """I1 = Re F^-1(F(I0) CTF Env) for one orientation and a list of CTF tables K [C][N][N]; returns [C][N][N]."""
    if model["kind"] == "atoms":
        F0 = np.fft.fft2(project_atoms(model["xyz"], model["radius"], model["weight"], q, N, px, int(model.get("Kq", 4))))
    else:
        F0 = fourier_slice(model["V"], model["voxel_A"], q)
    return np.fft.ifft2(F0[None] * K, axes=(1, 2)).real


def _chunk(args):
    model, N, px, D, quats, ctfs, images, lp_orient, lp_ctf, o_begin, o_end, n_orient_total = args
    n, S1 = N * N, 2 * D + 1
    S = S1 * S1
    obs = np.asarray(images, dtype=np.float64)
    I = obs.shape[0]
    Co, Coo = obs.sum(axis=(1, 2)), (obs * obs).sum(axis=(1, 2))
    Oc = np.conj(np.fft.rfft2(obs))
    K = np.stack([ctf_env_table(N, px, *c) for c in ctfs])
    idx = np.arange(-D, D + 1) % N
    st = RunState(I)
    C = len(ctfs)
    logS = math.log(S)
    for o in range(o_begin, o_end):
        I1s = calc_image_fft(model, quats[o], K, N, px)
        for c in range(C):
            I1 = I1s[c]
            Cc, Ccc = float(I1.sum()), float((I1 * I1).sum())
            cco = np.fft.irfft2(Oc * np.fft.rfft2(I1)[None], s=(N, N))[:, idx][:, :, idx].reshape(I, S)     # [img][dy][dx]
            logw = (lp_orient[o] if lp_orient is not None else -math.log(n_orient_total)) + \
                   (lp_ctf[c] if lp_ctf is not None else -math.log(C)) - logS
            lp = log_post_c1(n, Co[:, None], Coo[:, None], Cc, Ccc, cco) + logw
            base = (o * C + c) * S
            for w in range(I):
                x = lp[w]
                # the terms of this pair, folded in loop order: log-sum-exp, largest and second largest, strict argmax
                k = int(np.argmax(x))                        # first maximum = lowest flat index among ties
                mx = x[k]
                if mx == -np.inf:                            # a grid point of weight zero (R7) adds nothing
                    continue
                if mx > st.m[w]:
                    st.s[w] = st.s[w] * math.exp(st.m[w] - mx) + float(np.exp(x - mx).sum()) if st.m[w] > -np.inf else float(np.exp(x - mx).sum())
                    st.m[w] = mx
                else:
                    st.s[w] += float(np.exp(x - st.m[w]).sum())
                part = np.partition(x, S - 2)[S - 2] if S > 1 else -np.inf                      # second largest of this pair
                if mx > st.best[w]:
                    st.second[w] = max(st.best[w], part)
                    st.best[w], st.best_flat[w] = mx, base + k
                else:
                    st.second[w] = max(st.second[w], mx)
    return st.m, st.s, st.best, st.second, st.best_flat


def merge(states):
    """Fold chunk states in chunk (= orientation) order: the same result as one pass over the whole grid."""
    m, s, best, second, flat = (np.array(x, copy=True) for x in states[0])
    for m2, s2, b2, sec2, f2 in states[1:]:
        M = np.maximum(m, m2)
        with np.errstate(invalid="ignore"):
            s = np.where(np.isfinite(M), s * np.exp(np.where(np.isfinite(m), m - M, -np.inf)) +
                         s2 * np.exp(np.where(np.isfinite(m2), m2 - M, -np.inf)), 0.0)
        m = M
        newer = b2 > best                                    # strict: an equal term of a later chunk has the higher flat index
        second = np.where(newer, np.maximum(best, sec2), np.maximum(second, b2))
        flat = np.where(newer, f2, flat)
        best = np.where(newer, b2, best)
    st = RunState(len(m))
    st.m, st.s, st.best, st.second, st.best_flat = m, s, best, second, flat.astype(np.int64)
    return st


def run_model_fft(model, N, px, D, quats, ctfs, images, lp_orient=None, lp_ctf=None, workers=None, chunk=None):
    """Eq. 9 on the grid for ONE model, every image, all orientations x CTFs x shifts; returns a RunState like run_model.
    The orientation loop is cut into chunks that worker processes (spawned) take; states are merged in orientation order."""
    model = prepare_model(model)
    quats = np.ascontiguousarray(quats, dtype=np.float64)
    ctfs = np.ascontiguousarray(ctfs, dtype=np.float64)
    O = len(quats)
    if workers is None:
        workers = min(os.cpu_count() or 1, 32)
    if chunk is None:
        chunk = max(1, -(-O // (4 * workers)))
    jobs = [(model, N, px, D, quats, ctfs, images, lp_orient, lp_ctf, a, min(a + chunk, O), O) for a in range(0, O, chunk)]
    if workers <= 1 or len(jobs) == 1:
        return merge([_chunk(j) for j in jobs])
    import multiprocessing as mp
    from concurrent.futures import ProcessPoolExecutor
    with ProcessPoolExecutor(max_workers=workers, mp_context=mp.get_context("spawn")) as ex:
        return merge(list(ex.map(_chunk, jobs)))


def shift_map_fft(image, I1, D, logw):
    """log P(C1) + logw for every shift of one pair through the FFT route: [dy+D][dx+D] (the tier-C twin of shift_map)."""
    obs = np.asarray(image, dtype=np.float64)
    I1 = np.asarray(I1, dtype=np.float64)
    N = obs.shape[0]
    idx = np.arange(-D, D + 1) % N
    cco = np.fft.irfft2(np.conj(np.fft.rfft2(obs)) * np.fft.rfft2(I1), s=(N, N))[idx][:, idx]
    return log_post_c1(N * N, obs.sum(), (obs * obs).sum(), float(I1.sum()), float((I1 * I1).sum()), cco) + logw
