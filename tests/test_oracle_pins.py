"""Pins for the FP64 oracle: every check compares `oracle/` with something that is NOT the oracle --
a library routine, a closed form, a hand-built case, brute force, or numerical quadrature of Eq. 8.
(CPU only; `-m "not gpu"`.)  Citations: P:<line> of PAPER.md, R<k> of DESIGN.md section 3."""
import math

import numpy as np
import pytest

import oracle
import bioem_workloads as W
from bioem_workloads import simulate

RNG = np.random.default_rng(20161)


# ------------------------------------------------------------------ DFT (Eqs. 2-3, R3)
@pytest.mark.parametrize("N", [6, 8, 14])
def test_dft2_matches_library_fft(N):
    x = RNG.normal(size=(N, N)) + 1j * RNG.normal(size=(N, N))
    assert np.allclose(oracle.dft2(x, -1), np.fft.fft2(x), atol=1e-11)
    assert np.allclose(oracle.dft2(x, +1, 1.0 / N ** 2), np.fft.ifft2(x), atol=1e-12)


def test_plancherel():
    # C_oo ~ sum |F(I)|^2
    x = RNG.normal(size=(12, 12))
    F = oracle.dft2(x)
    assert math.isclose((x ** 2).sum(), (np.abs(F) ** 2).sum() / x.size, rel_tol=1e-12)


def test_dft3_matches_library():
    rho = RNG.normal(size=(6, 6, 6))
    assert np.allclose(oracle.dft3(rho), np.fft.fftn(rho), atol=1e-10)


# ------------------------------------------------------------------ cross-correlation (Eq. 7 / 11 / 12; R4, R5)
def test_cross_corr_delta_images_pin_the_shift_sign():
    # I_obs = delta at (j0,k0), I1 = delta at (j1,k1):  C_co(d) = sum_r I_obs(r) I1(r+d) = 1 iff r0 + d == r1 (mod N)
    N, D = 8, 3
    a = np.zeros((N, N)); b = np.zeros((N, N))
    j0, k0, j1, k1 = 2, 5, 4, 3            # x = j (fast index), y = k
    a[k0, j0] = 1.0; b[k1, j1] = 1.0
    C = oracle.cross_corr_direct(a, b, D)
    want = np.zeros((2 * D + 1, 2 * D + 1)); want[(k1 - k0) + D, (j1 - j0) + D] = 1.0     # dy = -2, dx = +2
    assert np.array_equal(C, want)
    # wrap-around (R5): delta near the border
    a[:] = 0; b[:] = 0; a[7, 7] = 1.0; b[1, 0] = 1.0     # dx = 0-7 = +1 (mod 8), dy = 1-7 = +2 (mod 8)
    C = oracle.cross_corr_direct(a, b, D)
    assert C[2 + D, 1 + D] == 1.0 and C.sum() == 1.0


@pytest.mark.parametrize("N,D", [(8, 3), (6, 2), (7, 3)])
def test_direct_sum_equals_naive_dft_eq12(N, D):
    # north_star check 1: the FFT-free correlation equals a naive DFT evaluation of Eq. 12 on tiny images
    a, b = RNG.normal(size=(N, N)), RNG.normal(size=(N, N))
    C = oracle.cross_corr_direct(a, b, D)
    assert np.allclose(C, oracle.cross_corr_eq12(a, b, D), atol=1e-12)
    assert np.allclose(C, oracle.cross_corr_dft(a, b, D), atol=1e-12)                      # tier B
    # library routine: irfft2(conj(A) B)[dy mod N, dx mod N]
    lib = np.fft.ifft2(np.conj(np.fft.fft2(a)) * np.fft.fft2(b)).real
    idx = np.arange(-D, D + 1) % N
    assert np.allclose(C, lib[np.ix_(idx, idx)], atol=1e-12)


def test_tier_b_matches_direct_on_a_real_pair():
    wl = W.build_workload("tiny_mini")
    s = wl["spec"]
    I1 = oracle.calc_image(wl["models"][0], wl["quats"][1], wl["ctfs"][2], s.n_pix, s.pixel_A)
    img = wl["images"][0].astype(np.float64)
    A, B = oracle.cross_corr_direct(img, I1, s.max_shift), oracle.cross_corr_dft(img, I1, s.max_shift)
    assert np.abs(A - B).max() <= 1e-9 * np.abs(A).max()


def test_shift_of_observed_image_moves_the_map():
    # d <-> rolling I_obs: I_obs'(r) = I_obs(r - e)  =>  C'(d) = C(d - e)... checked on the unpruned map
    N, D = 8, 4
    a, b = RNG.normal(size=(N, N)), RNG.normal(size=(N, N))
    C = oracle.cross_corr_direct(a, b, D)
    a2 = np.roll(a, shift=(1, 2), axis=(0, 1))         # a2[k][j] = a[k-1][j-2]
    C2 = oracle.cross_corr_direct(a2, b, D)
    # sum_r a(r - e) b(r + d) = sum_r a(r) b(r + d + e)  =>  C2(d) = C(d + e), e = (ex=2, ey=1)
    assert np.allclose(C2[0:2 * D, 0:2 * D - 1], C[1:2 * D + 1, 2:2 * D + 1], atol=1e-12)


# ------------------------------------------------------------------ closed form (stands in for Eq. S8; R1)
def _sums(obs, cal):
    return obs.size, obs.sum(), (obs ** 2).sum(), cal.sum(), (cal ** 2).sum(), (obs * cal).sum()


def _quadrature_log_marginal(obs, cal):
    """log of int dN dmu dlambda of Eq. 8 with I_cal = N*cal - mu (Eq. 7) and unit priors.
    The integrand is the raw sum of squares at every node; the completed squares only centre the grids."""
    n = obs.size
    Co, Coo, Cc, Ccc, Cco = obs.sum(), (obs ** 2).sum(), cal.sum(), (cal ** 2).sum(), (obs * cal).sum()
    A, B, Dd = Ccc - Cc ** 2 / n, Cco - Co * Cc / n, Coo - Co ** 2 / n
    E = Dd - B ** 2 / A
    Nstar = B / A
    u = np.linspace(math.log(2e-3 * math.sqrt(E / n)), math.log(5e2 * math.sqrt(E / n)), 1201)
    K = 201                                                                # survey 8(c): >= 200 nodes per Gaussian integral
    t = np.linspace(-12.0, 12.0, K)
    vals = np.empty_like(u)
    for i, lam in enumerate(np.exp(u)):
        Ng = Nstar + t * lam / math.sqrt(A)                               # [K]
        mustar = (Ng * Cc - Co) / n
        mug = mustar[:, None] + t[None, :] * lam / math.sqrt(n)           # [K_N][K_mu]
        resid = obs[None, None, :] - Ng[:, None, None] * cal[None, None, :] + mug[:, :, None]
        logL = -(resid ** 2).sum(-1) / (2 * lam * lam) - 0.5 * n * math.log(2 * math.pi * lam * lam)
        ref = logL.max()
        w = np.exp(logL - ref)
        inner = np.trapezoid(w, dx=(t[1] - t[0]) * lam / math.sqrt(n), axis=1)
        outer = np.trapezoid(inner, dx=(t[1] - t[0]) * lam / math.sqrt(A))
        vals[i] = math.log(outer) + ref + u[i]                            # d lambda = lambda du
    ref = vals.max()
    return math.log(np.trapezoid(np.exp(vals - ref), dx=u[1] - u[0])) + ref


@pytest.mark.parametrize("n", [9, 12, 16])
def test_closed_form_equals_quadrature_of_eq8(n):
    # north_star check 3
    rng = np.random.default_rng(100 + n)
    obs = rng.normal(size=n) * 1.7 + 0.4
    cal = rng.normal(size=n) * 0.6 - 0.2
    obs = obs + 0.8 * cal                      # some correlation
    c1 = oracle.log_post_c1(*_sums(obs, cal))
    c2 = oracle.log_post_c2(*_sums(obs, cal))
    quad = _quadrature_log_marginal(obs, cal)
    assert abs(c1 - c2) < 1e-10
    assert abs(c1 - quad) < 1e-8, (c1, quad)                     # survey 8(c): agree to <= 1e-8 in log


def test_eq8_function_matches_its_definition():
    rng = np.random.default_rng(5)
    obs, cal = rng.normal(size=10), rng.normal(size=10)
    Nn, mu, lam = 1.3, -0.2, 0.7
    want = -((obs - (Nn * cal - mu)) ** 2).sum() / (2 * lam ** 2) - 5 * math.log(2 * math.pi * lam ** 2)
    assert math.isclose(oracle.log_lik_eq8(obs, cal, Nn, mu, lam), want, rel_tol=1e-13)


def test_const_n_closed_form():
    # const(n) = -((n-2)/2) log 2pi + ((n-5)/2) log 2 + lgamma((n-3)/2); n = 5 -> lgamma(1) = 0
    assert math.isclose(oracle.const_n(5), -1.5 * math.log(2 * math.pi), rel_tol=1e-14)
    assert math.isclose(oracle.const_n(7), -2.5 * math.log(2 * math.pi) + math.log(2.0), rel_tol=1e-14)   # lgamma(2)=0


def test_closed_form_invariances():
    rng = np.random.default_rng(77)
    n = 64
    obs, cal = rng.normal(size=n) + 2.0, rng.normal(size=n)
    base = oracle.log_post_c1(*_sums(obs, cal))
    al, be, ga, de = 3.7, -11.0, -0.25, 5.0
    # I_obs -> alpha I_obs + beta : log P shifts by -(n-3) log|alpha|
    assert math.isclose(oracle.log_post_c1(*_sums(al * obs + be, cal)), base - (n - 3) * math.log(abs(al)), abs_tol=1e-9)
    # I1 -> gamma I1 + delta : log P shifts by -log|gamma|   (N < 0 allowed, R1)
    assert math.isclose(oracle.log_post_c1(*_sums(obs, ga * cal + de)), base - math.log(abs(ga)), abs_tol=1e-9)
    # joint permutation of pixels (e.g. a joint circular shift) changes nothing
    p = rng.permutation(n)
    assert math.isclose(oracle.log_post_c1(*_sums(obs[p], cal[p])), base, abs_tol=1e-10)


def test_c1_c2_agree_at_workload_scale():
    wl = W.build_workload("tiny_mini")
    s = wl["spec"]
    I1 = oracle.calc_image(wl["models"][0], wl["quats"][0], wl["ctfs"][0], s.n_pix, s.pixel_A)
    img = wl["images"][0].astype(np.float64)
    n, Co, Coo, Cc, Ccc, _ = _sums(img.ravel(), I1.ravel())
    C = oracle.cross_corr_direct(img, I1, 2)
    for cco in C.ravel():
        assert abs(oracle.log_post_c1(n, Co, Coo, Cc, Ccc, cco) - oracle.log_post_c2(n, Co, Coo, Cc, Ccc, cco)) < 1e-8


# ------------------------------------------------------------------ projection (Eq. 1; R10-R12)
def test_projection_total_mass_converges_to_sum_of_weights():
    rng = np.random.default_rng(3)
    xyz = rng.uniform(-20, 20, size=(50, 3)); rad = rng.uniform(1.0, 2.0, 50); wt = rng.uniform(1, 8, 50)
    q = np.array([0.3, -0.5, 0.2, 0.78]); q /= np.linalg.norm(q)
    m4 = oracle.project_atoms(xyz, rad, wt, q, 64, 1.0, 4).sum()
    m32 = oracle.project_atoms(xyz, rad, wt, q, 64, 1.0, 32).sum()
    assert abs(m4 / wt.sum() - 1) < 0.04
    assert abs(m32 / wt.sum() - 1) < 2e-3


def test_projection_single_sphere_values():
    # sphere inside one pixel: that pixel holds all the mass; big sphere: centre pixel ~ chord * px^2 * density
    N, px = 16, 4.0
    I0 = oracle.project_atoms([[0.3, -0.2, 5.0]], [1.0], [2.5], [1, 0, 0, 0], N, px, 64)
    assert abs(I0[N // 2, N // 2] - 2.5) < 5e-3 and abs(I0.sum() - I0[N // 2, N // 2]) < 1e-12
    R = 30.0
    I0 = oracle.project_atoms([[0.0, 0.0, 0.0]], [R], [1.0], [1, 0, 0, 0], 64, 1.0, 8)
    assert math.isclose(I0[32, 32], 2 * R / (4 / 3 * math.pi * R ** 3), rel_tol=2e-4)
    # 4-fold symmetric footprint about pixel (N/2, N/2) (R11)
    assert np.allclose(I0[32 - 5:32 + 6, 32 - 5:32 + 6], I0[32 - 5:32 + 6, 32 - 5:32 + 6].T, atol=1e-15)
    assert np.allclose(I0[32 - 5:32 + 6, 32 - 5:32 + 6], I0[32 - 5:32 + 6, 32 - 5:32 + 6][::-1, ::-1], atol=1e-15)


def test_projection_rotations():
    rng = np.random.default_rng(4)
    xyz = rng.uniform(-10, 10, size=(30, 3)); rad = np.full(30, 1.5); wt = np.ones(30)
    N, px = 32, 2.0
    I_id = oracle.project_atoms(xyz, rad, wt, [1, 0, 0, 0], N, px)
    # 180 deg about z: (x,y) -> (-x,-y): I0(j,k) -> I0(N-j, N-k)  (indices mod N; atoms are away from the border)
    I_z180 = oracle.project_atoms(xyz, rad, wt, [0, 0, 0, 1], N, px)
    idx = (-np.arange(N)) % N
    assert np.allclose(I_z180, I_id[np.ix_(idx, idx)], atol=1e-13)
    # active rotation (R12): +90 deg about z sends x -> y.  An atom at (+6,0,0) must land at y = +6 -> k = N/2 + 3
    I = oracle.project_atoms([[6.0, 0, 0]], [1.0], [1.0], [math.cos(math.pi / 4), 0, 0, math.sin(math.pi / 4)], N, px)
    k, j = np.unravel_index(np.argmax(I), I.shape)
    assert (j, k) == (N // 2, N // 2 + 3)
    # projection along z' : rotating about x by +90 deg sends y -> z (drops out) and z -> -y
    I = oracle.project_atoms([[0, 0, 8.0]], [1.0], [1.0], [math.cos(math.pi / 4), math.sin(math.pi / 4), 0, 0], N, px)
    k, j = np.unravel_index(np.argmax(I), I.shape)
    assert (j, k) == (N // 2, N // 2 - 4)
    # quaternion -> matrix against the Euler ZYZ product R = Rz(a) Ry(b) Rz(g)
    a, b, g = 0.4, 1.1, -2.0
    def rz(t): return np.array([[math.cos(t), -math.sin(t), 0], [math.sin(t), math.cos(t), 0], [0, 0, 1]])
    def ry(t): return np.array([[math.cos(t), 0, math.sin(t)], [0, 1, 0], [-math.sin(t), 0, math.cos(t)]])
    assert np.allclose(oracle.quat_to_matrix(W.euler_zyz_to_quat(a, b, g)), rz(a) @ ry(b) @ rz(g), atol=1e-14)


# ------------------------------------------------------------------ CTF (Eqs. 4-6; R8, R9)
def test_ctf_special_cases():
    rng = np.random.default_rng(8)
    I0 = rng.normal(size=(8, 8))
    # "CTF-free" (a=0, A=1, b=0): CTF Env == -1  ->  I1 = -I0  (R9)
    assert np.allclose(oracle.apply_ctf(I0, 1.5, 0.0, 1.0, 0.0), -I0, atol=1e-13)
    # A = 0: pure sine, zeros at a s^2/2 = m pi
    a = 31.0
    for m in (1, 2, 3):
        assert abs(oracle.ctf_env(2 * m * math.pi / a, a, 0.0, 0.0)) < 1e-13
    # s = 0: CTF = -A
    assert math.isclose(oracle.ctf_env(0.0, a, 0.1, 0.7), -0.1)
    # envelope
    assert math.isclose(oracle.ctf_env(3.0, 0.0, 1.0, 0.4), -math.exp(-0.6), rel_tol=1e-14)


def test_eq5_equals_eq6_psf_convolution():
    rng = np.random.default_rng(9)
    I0 = rng.normal(size=(8, 8))
    a, A, b = 9.0, 0.2, 0.8
    assert np.allclose(oracle.apply_ctf(I0, 1.5, a, A, b), oracle.apply_psf_realspace(I0, 1.5, a, A, b), atol=1e-12)


def test_ctf_matches_library_fft_route():
    rng = np.random.default_rng(10)
    N, px = 12, 1.5
    I0 = rng.normal(size=(N, N))
    a, A, b = 31.3, 0.1, 0.63
    want = np.fft.irfft2(np.fft.rfft2(I0) * simulate.ctf_image(N, px, a, A, b), s=(N, N))
    assert np.allclose(oracle.apply_ctf(I0, px, a, A, b), want, atol=1e-12)


def test_defocus_constants_r8_r9():
    # lambda_e(300 kV) = 0.019687 A; 1 um -> a = 31.33 A^2; B = 50 A^2 -> b = 0.633 A^2
    assert abs(W.generate.electron_wavelength_A(300.0) - 0.019687) < 1e-6
    a, b = W.ctf_from_defocus(1.0, 50.0, 300.0)
    assert abs(a - 31.33) < 5e-3 and abs(b - 0.6333) < 1e-4


# ------------------------------------------------------------------ density model / Fourier slice (R21)
def _blob_map(n, vox, centres, sig):
    ax = (np.arange(n) - n // 2) * vox
    Z, Y, X = np.meshgrid(ax, ax, ax, indexing="ij")
    rho = np.zeros((n, n, n))
    for c in centres:
        rho += np.exp(-0.5 * ((X - c[0]) ** 2 + (Y - c[1]) ** 2 + (Z - c[2]) ** 2) / sig ** 2)
    return rho


def test_fourier_slice_identity_is_dft_of_z_sum():
    n, vox = 16, 1.5
    rho = _blob_map(n, vox, [[2.0, -1.0, 3.0], [-3.0, 2.5, -1.0]], 2.0)
    F = oracle.fourier_slice(oracle.dft3(rho), vox, [1, 0, 0, 0])
    want = np.fft.fft2(rho.sum(0) * vox)
    h = n // 2
    keep = np.ones((n, n), bool); keep[h, :] = False; keep[:, h] = False
    assert np.allclose(F[keep], want[keep], atol=1e-10)
    assert np.all(F[~keep] == 0)


def test_fourier_slice_axis_rotation_is_index_permutation():
    n, vox = 16, 1.0
    rho = _blob_map(n, vox, [[2.0, -1.0, 3.0], [-3.0, 2.0, -1.0], [0.5, 3.0, 2.0]], 1.5)
    V = oracle.dft3(rho)
    # +90 deg about z, active: rho'(x,y,z) = rho(y,-x,z).  Projection image I'(x,y) = I(y,-x).
    q = [math.cos(math.pi / 4), 0, 0, math.sin(math.pi / 4)]
    F_rot, F_id = oracle.fourier_slice(V, vox, q), oracle.fourier_slice(V, vox, [1, 0, 0, 0])
    # I'(x,y) = I(y,-x)  =>  F'(l', m') = F(m', -l')   (arrays are [y-frequency][x-frequency]).
    # sqrt(1/2) is not exact, so bins with |l'| or |m'| = n/2 - 1 may fall just outside the |k_i| <= n/2 - 1 rule: skip them
    h = n // 2
    for ls in range(-h + 2, h - 1):
        for ms in range(-h + 2, h - 1):
            assert abs(F_rot[ms % n, ls % n] - F_id[(-ls) % n, ms % n]) < 1e-9


def test_fourier_slice_general_orientation_vs_analytic_blobs():
    # loose pin (interpolation error, not a parity bound): projected Gaussians at actively rotated centres (R12)
    n, vox, sig = 32, 1.5, 3.0
    centres = np.array([[5.0, -3.0, 4.0], [-6.0, 2.0, -2.0], [1.0, 7.0, 3.0]])
    rho = _blob_map(n, vox, centres, sig)
    q = W.euler_zyz_to_quat(0.7, 1.0, -0.4)
    img = -oracle.apply_ctf_spectrum(oracle.fourier_slice(oracle.dft3(rho), vox, q), vox, 0.0, 1.0, 0.0)
    R = oracle.quat_to_matrix(q)
    rc = centres @ R.T
    ax = (np.arange(n) - n // 2) * vox
    Y, X = np.meshgrid(ax, ax, indexing="ij")
    want = np.zeros((n, n))
    for c in rc:
        want += math.sqrt(2 * math.pi) * sig * np.exp(-0.5 * ((X - c[0]) ** 2 + (Y - c[1]) ** 2) / sig ** 2)
    assert np.corrcoef(img.ravel(), want.ravel())[0, 1] > 0.99
    # the transposed (passive) convention must NOT fit
    wrong = np.zeros((n, n))
    for c in centres @ R:
        wrong += math.sqrt(2 * math.pi) * sig * np.exp(-0.5 * ((X - c[0]) ** 2 + (Y - c[1]) ** 2) / sig ** 2)
    assert np.corrcoef(img.ravel(), wrong.ravel())[0, 1] < 0.9


def _multiaffine_spectrum(n, coef):
    """A 3-D spectrum whose CENTRED form Vc(k) = a + i b.k + c kx ky + i d kx ky kz (k = signed frequencies) is
    multi-affine in k, hence reproduced EXACTLY by trilinear interpolation at any point; Hermitian (even real part, odd
    imaginary part).  Returned uncentred, V(k) = (-1)^(kx+ky+kz) Vc(k), array [kz][ky][kx]: what R21 interpolates."""
    a, b, c, d = coef
    ks = np.fft.fftfreq(n, 1.0 / n)                        # signed frequencies of the array indices (Nyquist = -n/2)
    KZ, KY, KX = np.meshgrid(ks, ks, ks, indexing="ij")
    Vc = a + 1j * (b[0] * KX + b[1] * KY + b[2] * KZ) + c * KX * KY + 1j * d * KX * KY * KZ
    return np.where((KX + KY + KZ) % 2 == 0, 1.0, -1.0) * Vc


def _multiaffine_slice(n, vox, coef, R):
    """The central section of that spectrum written out from R21's definition (no interpolation anywhere): the value of
    Vc at R^T (l, m, 0), times (-1)^(l+m) voxel, zero outside |k_i| <= n/2 - 1 and on the 2-D Nyquist bins."""
    a, b, c, d = coef
    h = n // 2
    F = np.zeros((n, n), complex)
    for ms in range(-h + 1, h):
        for ls in range(-h + 1, h):
            k = R.T @ np.array([ls, ms, 0.0])
            if np.all(np.abs(k) <= h - 1):
                v = a + 1j * (b @ k) + c * k[0] * k[1] + 1j * d * k[0] * k[1] * k[2]
                F[ms % n, ls % n] = (-1.0) ** (ls + ms) * vox * v
    return F


@pytest.mark.parametrize("seed", range(6))
def test_fourier_slice_general_orientation_is_exact_on_multiaffine_spectra(seed):
    # The tight pin at GENERAL orientations (R21): trilinear interpolation reproduces a multi-affine function exactly, so the
    # oracle's slice must equal the closed form element by element.  A nearest-neighbour or mis-weighted interpolation, a
    # transposed rotation, a wrong corner index, sign factor, voxel factor, cut-off rule or Hermitian completion fails this.
    rng = np.random.default_rng(4100 + seed)
    n, vox = 16, 1.3
    coef = (rng.normal(), rng.normal(size=3), rng.normal(), rng.normal())
    q = rng.normal(size=4)
    q /= np.linalg.norm(q)
    R = oracle.quat_to_matrix(q)
    got = oracle.fourier_slice(_multiaffine_spectrum(n, coef), vox, q)
    want = _multiaffine_slice(n, vox, coef, R)
    h = n // 2
    # points whose rotated coordinate lies within rounding of the cut-off |k_i| = n/2 - 1 may fall on either side
    edge = np.zeros((n, n), bool)
    for ms in range(-h + 1, h):
        for ls in range(-h + 1, h):
            k = R.T @ np.array([ls, ms, 0.0])
            edge[ms % n, ls % n] = np.any(np.abs(np.abs(k) - (h - 1)) < 1e-9)
    scale = np.abs(want).max()
    assert scale > 1.0
    assert np.abs(got - want)[~edge].max() < 1e-12 * scale
    # the passive (transposed) convention and a nearest-neighbour section must NOT fit
    assert np.abs(got - _multiaffine_slice(n, vox, coef, R.T))[~edge].max() > 1e-3 * scale


def test_fourier_slice_exact_index_permutations():
    # rotations that map the grid onto itself (interpolation weights 0 / 1): +90 deg about x, +90 deg about y, and 120 deg
    # about the body diagonal (q = (1,1,1,1)/2, exact in binary: R is the cyclic permutation x -> y -> z -> x)
    n, vox = 16, 1.0
    rho = _blob_map(n, vox, [[2.0, -1.0, 3.0], [-3.0, 2.0, -1.0], [0.5, 3.0, 2.0]], 1.5)
    V = oracle.dft3(rho)
    h = n // 2
    idx = np.arange(n)
    neg = (n - idx) % n                                   # index of the coordinate -(i - n/2) under the periodic grid

    def check(q, rot_rho):
        # rot_rho = rho'(r) = rho(R^-1 r) resampled on the grid (an index permutation); its z-sum is the projection (R12)
        want = np.fft.fft2(rot_rho.sum(0) * vox)
        got = oracle.fourier_slice(V, vox, q)
        for ls in range(-h + 2, h - 1):                   # 1/sqrt(2) is not exact: skip the bins next to the cut-off
            for ms in range(-h + 2, h - 1):
                assert abs(got[ms % n, ls % n] - want[ms % n, ls % n]) < 1e-9
    c, s_ = math.cos(math.pi / 4), math.sin(math.pi / 4)
    # Rx(+90): r' = (x, -z, y), R^-1 r = (x, z, -y): rho'[z][y][x] = rho[z' = -y][y' = z][x]
    check([c, s_, 0, 0], rho[neg][:, idx][:, :, idx].transpose(1, 0, 2))
    # Ry(+90): r' = (z, y, -x), R^-1 r = (-z, y, x): rho'[z][y][x] = rho[z' = x][y][x' = -z]
    check([c, 0, s_, 0], rho[:, :, neg].transpose(2, 1, 0))
    # 120 deg about (1,1,1): r' = (z, x, y), R^-1 r = (y, z, x): rho'[z][y][x] = rho[z' = x][y' = z][x' = y]
    check([0.5, 0.5, 0.5, 0.5], rho.transpose(1, 2, 0))


# ------------------------------------------------------------------ real-space, cropping displacement variant (R25)
def test_cropped_sums_delta_images_do_not_wrap():
    # obs = delta at (k0, j0), calc = delta at (k1, j1): C_co(d) = 1 exactly where (k0, j0) + d = (k1, j1), INSIDE the box only
    N, D = 8, 3
    obs = np.zeros((N, N)); obs[1, 6] = 1.0
    cal = np.zeros((N, N)); cal[3, 7] = 2.5
    cco, cc, ccc = oracle.cropped_sums(obs, cal, D)
    want = np.zeros((2 * D + 1, 2 * D + 1)); want[2 + D, 1 + D] = 2.5          # d = (dx, dy) = (+1, +2)
    assert np.array_equal(cco, want)
    # a pair that only meets through the border: circular (R5) finds it at d = (+2, 0), the cropping variant does not
    cal2 = np.zeros((N, N)); cal2[1, 0] = 1.0
    circ = oracle.cross_corr_direct(obs, cal2, D)
    crop, _, _ = oracle.cropped_sums(obs, cal2, D)
    assert circ[0 + D, 2 + D] == 1.0 and np.all(crop == 0.0)
    # C_c(d), C_cc(d): the delta of the calculated image at column 7 is pushed out of the box by any dx < 0 ... no: I_d(r) = I1(r+d)
    # keeps pixel p = r + d of I1 iff r = p - d is inside the box: column 7 survives iff 0 <= 7 - dx <= 7, i.e. dx >= 0
    for dy in range(-D, D + 1):
        for dx in range(-D, D + 1):
            inside = 0 <= 7 - dx < N and 0 <= 3 - dy < N
            assert cc[dy + D, dx + D] == (2.5 if inside else 0.0) and ccc[dy + D, dx + D] == (6.25 if inside else 0.0)


def test_cropped_sums_equal_explicit_zero_padded_shift():
    # brute force: build I_d(r) = I1(r + d) with zeros where r + d leaves the box, as an array, and take plain numpy sums
    rng = np.random.default_rng(77)
    N, D = 7, 2
    obs, cal = rng.normal(size=(N, N)), rng.normal(size=(N, N))
    cco, cc, ccc = oracle.cropped_sums(obs, cal, D)
    pad = np.zeros((N + 2 * D, N + 2 * D)); pad[D:D + N, D:D + N] = cal
    for dy in range(-D, D + 1):
        for dx in range(-D, D + 1):
            Id = pad[D + dy:D + dy + N, D + dx:D + dx + N]                       # Id[k][j] = cal[k + dy][j + dx] or 0
            assert abs(cco[dy + D, dx + D] - (obs * Id).sum()) < 1e-12
            assert abs(cc[dy + D, dx + D] - Id.sum()) < 1e-12 and abs(ccc[dy + D, dx + D] - (Id * Id).sum()) < 1e-12


def test_cropping_variant_equals_circular_variant_when_nothing_reaches_the_border():
    # the two variants differ only in what happens at the borders: with the calculated image supported more than D
    # pixels away from them, Eq. 9 on the grid is the same number either way (tier 2 vs tier 0 of the same loop nest)
    spec = W.get_spec("tiny_mini")
    wl = W.build_workload(spec)
    s = wl["spec"]
    m = dict(wl["models"][0]); m["xyz"] = np.asarray(m["xyz"]) * 0.5             # 15 A ball in a 128 A box: far from the borders
    a = oracle.run_model(m, s.n_pix, s.pixel_A, 3, wl["quats"][:2], wl["ctfs"][:1] * [0, 1, 0] + [0, 0, 0], wl["images"][:2], tier=0)
    b = oracle.run_model(m, s.n_pix, s.pixel_A, 3, wl["quats"][:2], wl["ctfs"][:1] * [0, 1, 0] + [0, 0, 0], wl["images"][:2], tier=2)
    assert np.abs(a.log_posterior() - b.log_posterior()).max() < 1e-9 and np.array_equal(a.best_flat, b.best_flat)
    # ... and differ once the CTF spreads the calculated image over the whole box
    a = oracle.run_model(m, s.n_pix, s.pixel_A, 3, wl["quats"][:2], wl["ctfs"][:1], wl["images"][:2], tier=0)
    b = oracle.run_model(m, s.n_pix, s.pixel_A, 3, wl["quats"][:2], wl["ctfs"][:1], wl["images"][:2], tier=2)
    assert np.abs(a.log_posterior() - b.log_posterior()).max() > 1e-6


# ------------------------------------------------------------------ synthetic map for a parameter set theta
def test_synthetic_map_displacement_is_the_one_of_the_cross_correlation():
    # sum_r obs(r) S(r) with N = 1, mu = 0 IS C_co(d) of bo_cross_corr_direct (wrapping, R5) / bo_cropped_sums (cropping, R25):
    # a flipped sign or swapped axis of d in either place breaks this
    rng = np.random.default_rng(5)
    N, D = 9, 3
    obs, cal = rng.normal(size=(N, N)), rng.normal(size=(N, N))
    circ = oracle.cross_corr_direct(obs, cal, D)
    crop, _, _ = oracle.cropped_sums(obs, cal, D)
    for dy in range(-D, D + 1):
        for dx in range(-D, D + 1):
            S, n_, mu = oracle.synthetic_map(cal, dx, dy)
            assert (n_, mu) == (1.0, 0.0) and abs((obs * S).sum() - circ[dy + D, dx + D]) < 1e-12
            Sc, _, _ = oracle.synthetic_map(cal, dx, dy, crop=True)
            assert abs((obs * Sc).sum() - crop[dy + D, dx + D]) < 1e-12
    # by hand: a single pixel of the calculated image at (k, j) = (3, 7), displaced by (dx, dy) = (+1, +2), appears at (1, 6);
    # displaced by dx = -2 it leaves the 9-pixel box on the right: wrapped to column 0, cropped away
    cal = np.zeros((N, N)); cal[3, 7] = 2.5
    want = np.zeros((N, N)); want[1, 6] = 2.5
    assert np.array_equal(oracle.synthetic_map(cal, 1, 2)[0], want) and np.array_equal(oracle.synthetic_map(cal, 1, 2, crop=True)[0], want)
    want = np.zeros((N, N)); want[3, 0] = 2.5
    assert np.array_equal(oracle.synthetic_map(cal, -2, 0)[0], want) and not oracle.synthetic_map(cal, -2, 0, crop=True)[0].any()


def test_synthetic_map_normalisation_and_offset_maximise_eq8():
    rng = np.random.default_rng(6)
    N = 10
    cal = rng.normal(size=(N, N))
    Id = oracle.synthetic_map(cal, 2, -1)[0]
    # exact recovery: an image that IS I_cal of Eq. 7 with N = 2.5, mu = 0.7 (the offset is SUBTRACTED there)
    S, n_, mu = oracle.synthetic_map(cal, 2, -1, obs=2.5 * Id - 0.7)
    assert abs(n_ - 2.5) < 1e-12 and abs(mu - 0.7) < 1e-12 and np.abs(S - (2.5 * Id - 0.7)).max() < 1e-12
    # library routine: linear least squares of obs on (I_d, 1)
    obs = 1.7 * Id + 0.3 + rng.normal(size=(N, N))
    S, n_, mu = oracle.synthetic_map(cal, 2, -1, obs=obs)
    ref = np.linalg.lstsq(np.stack([Id.ravel(), np.ones(N * N)], axis=1), obs.ravel(), rcond=None)[0]
    assert abs(n_ - ref[0]) < 1e-10 and abs(mu + ref[1]) < 1e-10 and np.abs(S - (n_ * Id - mu)).max() < 1e-12
    # the paper's likelihood (Eq. 8, bo_log_lik_eq8) is largest there, at any lambda
    for lam in (0.4, 1.3):
        top = oracle.log_lik_eq8(obs, Id, n_, mu, lam)
        for dn, dm in ((1e-3, 0), (-1e-3, 0), (0, 1e-3), (0, -1e-3), (7e-4, -7e-4)):
            assert oracle.log_lik_eq8(obs, Id, n_ + dn, mu + dm, lam) < top


# ------------------------------------------------------------------ Eq. 9 on the grid (R7, R15, R16)
def test_planted_truth_is_the_argmax():
    # north_star check 2: a noiseless, CTF-free image at a grid orientation and shift scores its maximum exactly there
    spec = W.get_spec("tiny")
    model = W.make_atom_model(spec)
    quats = W.generate.orientation_grid(spec)[::5]           # 13 orientations
    ctfs = np.array([[0.0, 1.0, 0.0]])
    D, N, px = 3, spec.n_pix, spec.pixel_A
    o_true, dx, dy = 7, 2, -3
    I1 = oracle.calc_image(model, quats[o_true], ctfs[0], N, px)
    img = (1.7 * np.roll(I1, shift=(-dy, -dx), axis=(0, 1)) + 0.3).astype(np.float32)[None]
    st = oracle.run_model(model, N, px, D, quats, ctfs, img)
    o, c, bx, by = oracle.unflatten(st.best_flat, 1, D)
    assert (o[0], c[0], bx[0], by[0]) == (o_true, 0, dx, dy)
    assert st.best[0] - st.second[0] > 100.0


def test_log_sum_exp_equals_brute_force_and_chunking_is_exact():
    wl = W.build_workload("tiny_mini")
    s = wl["spec"]
    m = wl["models"][0]
    st = oracle.run_model(m, s.n_pix, s.pixel_A, s.max_shift, wl["quats"], wl["ctfs"], wl["images"])
    # brute force: all terms from per-pair maps, summed in long double
    logw = oracle.uniform_logw(len(wl["quats"]), len(wl["ctfs"]), s.max_shift)
    terms = [[] for _ in range(s.n_images)]
    for o, q in enumerate(wl["quats"]):
        for c, ctf in enumerate(wl["ctfs"]):
            I1 = oracle.calc_image(m, q, ctf, s.n_pix, s.pixel_A)
            for w in range(s.n_images):
                terms[w].append(oracle.shift_map(wl["images"][w], I1, s.max_shift, logw).ravel())
    for w in range(s.n_images):
        t = np.concatenate(terms[w]).astype(np.longdouble)
        want = float(t.max() + np.log(np.exp(t - t.max()).sum()))
        assert abs(st.log_posterior()[w] - want) < 1e-10
        assert st.best_flat[w] == int(np.argmax(t)) and st.best[w] == float(t.max())
    # chunked over orientations == one shot, bit for bit
    st2 = oracle.run_model(m, s.n_pix, s.pixel_A, s.max_shift, wl["quats"], wl["ctfs"], wl["images"], o_end=2)
    st2 = oracle.run_model(m, s.n_pix, s.pixel_A, s.max_shift, wl["quats"], wl["ctfs"], wl["images"], o_begin=2, state=st2)
    assert np.array_equal(st2.log_posterior(), st.log_posterior()) and np.array_equal(st2.best_flat, st.best_flat)
    # tier B agrees with the definition
    st3 = oracle.run_model(m, s.n_pix, s.pixel_A, s.max_shift, wl["quats"], wl["ctfs"], wl["images"], tier=1)
    assert np.abs(st3.log_posterior() - st.log_posterior()).max() < 1e-8
    assert np.array_equal(st3.best_flat, st.best_flat)


def test_equal_terms_sum_to_the_term():
    # R7: with uniform weights, identical terms -> LSE equals the term (weights sum to one)
    st = oracle.RunState(1)
    N = 8
    model = dict(kind="atoms", xyz=np.zeros((1, 3)), radius=np.array([3.0]), weight=np.array([1.0]), Kq=4)
    img = RNG.normal(size=(1, N, N)).astype(np.float32)
    # a sphere at the origin looks the same from every orientation about z; D = 0 -> one shift
    quats = np.array([[math.cos(t / 2), 0, 0, math.sin(t / 2)] for t in (0.0, math.pi / 2, math.pi, 3 * math.pi / 2)])
    st = oracle.run_model(model, N, 1.0, 0, quats, np.array([[0.0, 1.0, 0.0]]), img)
    one = oracle.run_model(model, N, 1.0, 0, quats[:1], np.array([[0.0, 1.0, 0.0]]), img)
    assert abs(st.log_posterior()[0] - one.log_posterior()[0]) < 1e-10
    assert st.best_flat[0] == 0            # exact ties keep the lowest flat index (R15)


# ------------------------------------------------------------------ stored fixtures (tests/golden/, each file cites its source)
GOLDEN = __import__("pathlib").Path(__file__).resolve().parent / "golden"


def _rows(name):
    return [ln for ln in (GOLDEN / name).read_text().splitlines() if ln.strip() and not ln.startswith("#")]


def test_golden_ctf_constants():
    g = {r.split()[0]: (float(r.split()[1]), float(r.split()[2])) for r in _rows("ctf_constants.txt")}
    for kv in (100, 200, 300):
        v, tol = g[f"lambda_A_{kv}kV"]
        assert abs(W.generate.electron_wavelength_A(float(kv)) - v) <= tol
    a, b = W.ctf_from_defocus(1.0, 50.0, 300.0)
    assert abs(a - g["a_A2_1um_300kV"][0]) <= g["a_A2_1um_300kV"][1]
    assert abs(b - g["b_A2_B50"][0]) <= g["b_A2_B50"][1]
    # ... and the oracle's CTF*Env (Eq. 4-5) at that (a, b): first zero of the pure phase CTF (A = 0) at a s^2 / 2 = pi
    s2 = 2 * np.pi / a
    assert abs(oracle.ctf_env(s2, a, 0.0, 0.0)) < 1e-12
    assert abs(oracle.ctf_env(s2, a, 0.0, b) / np.exp(-b * s2 / 2) ) < 1e-12
    assert abs(oracle.ctf_env(0.5 * s2, a, 0.0, b) - (-np.exp(-b * s2 / 4))) < 1e-12      # a s^2/2 = pi/2: -sin = -1 (R9 sign)


def test_golden_closed_form_vs_stored_quadrature_of_eq8():
    """(C1) and (C2) against the brute-force triple integral of the un-marginalised Eq. 8 on fixed inputs; the
    expected values were written by tests/golden/make_closed_form_golden.py, which imports nothing of the oracle."""
    rows = _rows("closed_form_quadrature.txt")
    assert len(rows) >= 3
    for r in rows:
        a, b, c = r.split("|")
        n = int(a.split()[0])
        io = np.array([float(x) for x in a.split()[1:]])
        ic = np.array([float(x) for x in b.split()])
        want = float(c)
        assert io.size == n and ic.size == n
        args = (n, io.sum(), (io * io).sum(), ic.sum(), (ic * ic).sum(), (io * ic).sum())
        assert abs(oracle.log_post_c1(*args) - want) <= 1e-9           # the fixture stores 10 decimals
        assert abs(oracle.log_post_c2(*args) - want) <= 1e-9


def test_orientation_posterior_pins():
    """P:225 'posterior as a function of orientation': (i) its log-sum-exp over orientations is the full log-posterior
    (Eq. 9 is a sum over the grid, so any partition of the grid adds up); (ii) each entry equals the log-sum-exp of the
    per-shift maps of that orientation's calculated images, built through a different oracle entry point (calc_image +
    shift_map) and numpy."""
    import bioem_workloads as W
    wl = W.build_workload("tiny_mini")
    s = wl["spec"]
    quats, ctfs, imgs = wl["quats"][:3], wl["ctfs"][:2], wl["images"][:2]
    D = 2
    po = oracle.orientation_log_posterior(wl["models"][0], s.n_pix, s.pixel_A, D, quats, ctfs, imgs)
    full = oracle.run_model(wl["models"][0], s.n_pix, s.pixel_A, D, quats, ctfs, imgs).log_posterior()
    m = po.max(axis=1)
    assert np.abs(m + np.log(np.exp(po - m[:, None]).sum(axis=1)) - full).max() <= 1e-10
    model = oracle.prepare_model(wl["models"][0])
    logw = oracle.uniform_logw(len(quats), len(ctfs), D)
    for i in range(len(imgs)):
        for o in range(len(quats)):
            maps = np.stack([oracle.shift_map(imgs[i], oracle.calc_image(model, quats[o], ctfs[c], s.n_pix, s.pixel_A), D, logw)
                             for c in range(len(ctfs))])
            mm = maps.max()
            assert abs(mm + math.log(np.exp(maps - mm).sum()) - po[i, o]) <= 1e-9


def test_ensemble_posterior_pins():
    """Eq. 10: against the product of weighted sums written out with plain exp on numbers small enough not to
    overflow; one model with weight 1 -> sum of its log-posteriors; a common offset c adds I*c; a zero-weight model drops out."""
    rng = np.random.default_rng(3)
    lp = rng.normal(0.0, 2.0, size=(5, 4))
    w = np.array([0.1, 0.2, 0.3, 0.4])
    tot, per = oracle.ensemble_log_posterior(lp, w)
    brute = 1.0
    for i in range(5):
        brute *= sum(w[m] * math.exp(lp[i, m]) for m in range(4))
    assert abs(tot - math.log(brute)) <= 1e-12 and abs(per.sum() - tot) <= 1e-12
    assert abs(oracle.ensemble_log_posterior(lp[:, :1], [1.0])[0] - lp[:, 0].sum()) <= 1e-12
    assert abs(oracle.ensemble_log_posterior(lp - 1e4, w)[0] - (tot - 5e4)) <= 1e-8
    assert abs(oracle.ensemble_log_posterior(lp, [0.5, 0.5, 0.0, 0.0])[0] - oracle.ensemble_log_posterior(lp[:, :2], [0.5, 0.5])[0]) <= 1e-12
    u, _ = oracle.ensemble_log_posterior(lp)
    assert abs(u - oracle.ensemble_log_posterior(lp, [0.25] * 4)[0]) <= 1e-12


# ------------------------------------------------------------------ tier C (oracle/fftgrid.py): the tier-A loop nest with numpy's FFT
@pytest.mark.parametrize("name", ["tiny", "small_mini", "paper_mini", "density_mini"])
def test_tier_c_matches_the_definition(name):
    """oracle/fftgrid.py replaces tier A's transforms and its direct correlation by numpy's FFT; everything it returns -- log-posterior,
    largest and second largest term, argmax -- must agree with tier A (direct summation, naive DFTs) on whole grids."""
    import bioem_workloads as W
    from oracle import fftgrid
    wl = W.build_workload(name)
    s = wl["spec"]
    a = oracle.run_model(wl["models"][0], s.n_pix, s.pixel_A, s.max_shift, wl["quats"], wl["ctfs"], wl["images"])
    b = fftgrid.run_model_fft(wl["models"][0], s.n_pix, s.pixel_A, s.max_shift, wl["quats"], wl["ctfs"], wl["images"], workers=1, chunk=2)
    assert np.abs(a.log_posterior() - b.log_posterior()).max() <= 1e-8
    assert np.abs(a.best - b.best).max() <= 1e-8 and np.abs(a.second - b.second).max() <= 1e-8
    assert np.array_equal(a.best_flat, b.best_flat)


def test_tier_c_pieces():
    from oracle import fftgrid
    # the CTF table against the C function, bin by bin (signed frequencies, Nyquist included)
    N, px, a, A, b = 8, 1.5, 31.33, 0.1, 0.633
    K = fftgrid.ctf_env_table(N, px, a, A, b)
    for m in range(N):
        for l in range(N):
            ls, ms = (l if l <= N // 2 else l - N), (m if m <= N // 2 else m - N)
            s2 = (2 * np.pi / (N * px)) ** 2 * (ls * ls + ms * ms)
            assert abs(K[m, l] - oracle.ctf_env(s2, a, A, b)) <= 1e-14
    # the vectorised closed form against bo_log_post_c1
    rng = np.random.default_rng(5)
    n = 64
    for _ in range(20):
        o, c = rng.normal(size=n), rng.normal(size=n)
        Co, Coo, Cc, Ccc, Cco = o.sum(), (o * o).sum(), c.sum(), (c * c).sum(), (o * c).sum()
        assert abs(float(fftgrid.log_post_c1(n, Co, Coo, Cc, Ccc, np.array([Cco]))[0]) - oracle.log_post_c1(n, Co, Coo, Cc, Ccc, Cco)) <= 1e-10
    # the shift-map twin against direct summation, wrap-around included
    img, I1 = rng.normal(size=(16, 16)).astype(np.float32), rng.normal(size=(16, 16))
    assert np.abs(fftgrid.shift_map_fft(img, I1, 5, -1.25) - oracle.shift_map(img, I1, 5, -1.25)).max() <= 1e-9


def test_zero_weight_grid_points_add_nothing():
    """R7: a grid point with log-prior -inf has weight zero in Eq. 9's sum -- the result equals the run on the grid without it,
    also when the excluded point comes first (the running log-sum-exp then starts from an empty sum)."""
    import bioem_workloads as W
    wl = W.build_workload("tiny_mini")
    s = wl["spec"]
    O, Cn = len(wl["quats"]), len(wl["ctfs"])
    rng = np.random.default_rng(3)
    lpo, lpc = np.log(rng.dirichlet(np.ones(O))), np.log(rng.dirichlet(np.ones(Cn)))
    lpo0, lpc0 = lpo.copy(), lpc.copy()
    lpo0[0] = -np.inf
    lpc0[0] = -np.inf
    a = oracle.run_model(wl["models"][0], s.n_pix, s.pixel_A, s.max_shift, wl["quats"], wl["ctfs"], wl["images"], lp_orient=lpo0, lp_ctf=lpc0)
    b = oracle.run_model(wl["models"][0], s.n_pix, s.pixel_A, s.max_shift, wl["quats"][1:], wl["ctfs"][1:], wl["images"],
                         lp_orient=lpo[1:], lp_ctf=lpc[1:])
    assert np.all(np.isfinite(a.log_posterior())) and np.abs(a.log_posterior() - b.log_posterior()).max() <= 1e-9
    oa, ca, dxa, dya = oracle.unflatten(a.best_flat, Cn, s.max_shift)
    ob, cb, dxb, dyb = oracle.unflatten(b.best_flat, Cn - 1, s.max_shift)
    assert np.array_equal(oa, ob + 1) and np.array_equal(ca, cb + 1) and np.array_equal(dxa, dxb) and np.array_equal(dya, dyb)
