"""ctypes binding with the same names as include/bioem.h.  PyTorch supplies device memory and the stream."""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_LIBPATH = _HERE / "libbioem_b200.so"
TOPK = 8

EXPORTED_SYMBOLS = [
    "bioem_create", "bioem_destroy", "bioem_last_error", "bioem_set_image_geometry", "bioem_clear_models",
    "bioem_add_model_atoms", "bioem_add_model_density", "bioem_set_orientations_quat", "bioem_set_ctf_grid",
    "bioem_ctf_from_defocus", "bioem_set_shift_range", "bioem_push_images", "bioem_run", "bioem_get_log_posterior",
    "bioem_get_best", "bioem_debug_calc_image", "bioem_debug_shift_map", "bioem_debug_shift_map_f64",
    "bioem_debug_log_posterior_f32", "bioem_get_timing", "bioem_get_launch_count", "bioem_measure_fp32_peak",
    "bioem_set_orientation_posterior", "bioem_get_orientation_log_posterior", "bioem_get_ensemble_log_posterior",
    "bioem_set_orientation_chunk", "bioem_debug_set_kernel", "bioem_get_run_plan", "bioem_invalidate_precompute",
    "bioem_set_orientation_slice", "bioem_run_partial", "bioem_get_partials_size", "bioem_export_partials", "bioem_merge_partials",
    "bioem_rescore_local", "bioem_export_rescore", "bioem_import_rescore", "bioem_finish", "bioem_set_displacement_variant",
    "bioem_get_synthetic_map", "bioem_noalloc_prepare", "bioem_ensemble_log_posterior_noalloc", "bioem_noalloc_last_error",
]
NOALLOC_MAX_IMG, NOALLOC_MAX_MODEL = 65536, 1024
KERNEL_AUTO, KERNEL_GENERIC, KERNEL_PK, KERNEL_C2, KERNEL_TM, KERNEL_DFT, KERNEL_REALSPACE = 0, 1, 2, 3, 4, 5, 6

_fp = C.POINTER(C.c_float)
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_lib = None


class BioEMError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"bioem error {code}: {msg}")
        self.code = code


def library_path() -> Path:
    return _LIBPATH


def lib():
    """Load the CUDA library.  Fails loudly when it has not been built: there is no fallback path."""
    global _lib
    if _lib is None:
        if not _LIBPATH.exists():
            raise ImportError(f"{_LIBPATH} is missing: run `python -m paper_1609_06634_b200.build` "
                              "(or __graft_entry__.build()); the CUDA extension is required, there is no CPU fallback")
        L = C.CDLL(str(_LIBPATH))
        L.bioem_last_error.restype = C.c_char_p
        L.bioem_last_error.argtypes = [C.c_void_p]
        L.bioem_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_void_p]
        L.bioem_destroy.argtypes = [C.c_void_p]
        L.bioem_set_image_geometry.argtypes = [C.c_void_p, C.c_int, C.c_float]
        L.bioem_clear_models.argtypes = [C.c_void_p]
        L.bioem_add_model_atoms.argtypes = [C.c_void_p, C.c_int, _fp, _fp, _fp, C.POINTER(C.c_int)]
        L.bioem_add_model_density.argtypes = [C.c_void_p, C.c_int, C.c_float, _fp, C.POINTER(C.c_int)]
        L.bioem_set_orientations_quat.argtypes = [C.c_void_p, C.c_int, _fp, _fp]
        L.bioem_set_ctf_grid.argtypes = [C.c_void_p, C.c_int, _fp, _fp, _fp, _fp]
        L.bioem_ctf_from_defocus.argtypes = [C.c_float, C.c_float, C.c_float, _fp, _fp]
        L.bioem_set_shift_range.argtypes = [C.c_void_p, C.c_int]
        L.bioem_push_images.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int]
        L.bioem_run.argtypes = [C.c_void_p]
        L.bioem_invalidate_precompute.argtypes = [C.c_void_p]
        L.bioem_set_orientation_slice.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.bioem_run_partial.argtypes = [C.c_void_p]
        L.bioem_get_partials_size.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int32)]
        L.bioem_export_partials.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.bioem_merge_partials.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int64, _ip, C.c_int]
        L.bioem_rescore_local.argtypes = [C.c_void_p]
        L.bioem_export_rescore.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.bioem_import_rescore.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.bioem_finish.argtypes = [C.c_void_p]
        L.bioem_set_displacement_variant.argtypes = [C.c_void_p, C.c_int]
        L.bioem_get_log_posterior.argtypes = [C.c_void_p, _dp]
        L.bioem_get_best.argtypes = [C.c_void_p, _ip, _ip, _ip, _ip, _dp]
        L.bioem_debug_calc_image.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, _fp]
        L.bioem_debug_shift_map.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, _dp]
        L.bioem_debug_shift_map_f64.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, _dp]
        L.bioem_debug_log_posterior_f32.argtypes = [C.c_void_p, _dp]
        L.bioem_get_timing.argtypes = [C.c_void_p, _dp, _dp]
        L.bioem_get_launch_count.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
        L.bioem_measure_fp32_peak.argtypes = [C.c_void_p, _dp, _dp]
        L.bioem_set_orientation_chunk.argtypes = [C.c_void_p, C.c_int]
        L.bioem_debug_set_kernel.argtypes = [C.c_void_p, C.c_int]
        L.bioem_get_run_plan.argtypes = [C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_int)]
        L.bioem_get_synthetic_map.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, _fp, _fp, _dp]
        L.bioem_noalloc_prepare.argtypes = [C.c_int]
        L.bioem_ensemble_log_posterior_noalloc.argtypes = [C.c_int, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.bioem_noalloc_last_error.argtypes = []
        for name in EXPORTED_SYMBOLS:
            if name != "bioem_last_error":
                getattr(L, name).restype = C.c_int
        L.bioem_noalloc_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def _f32(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a, a.ctypes.data_as(_fp)


def ctf_from_defocus(defocus_um, bfactor_A2, kV=300.0):
    a, b = C.c_float(), C.c_float()
    rc = lib().bioem_ctf_from_defocus(defocus_um, bfactor_A2, kV, C.byref(a), C.byref(b))
    if rc:
        raise BioEMError(rc, "bioem_ctf_from_defocus")
    return a.value, b.value


class BioEM:
    """One library context on one GPU.  Method names follow include/bioem.h without the ``bioem_`` prefix."""

    def __init__(self, device: int = 0, stream=None):
        self._h = C.c_void_p()
        self._L = lib()
        if stream is None:
            try:
                import torch
                if torch.cuda.is_available():
                    stream = torch.cuda.current_stream(device).cuda_stream
            except ImportError:
                stream = None
        rc = self._L.bioem_create(C.byref(self._h), device, C.c_void_p(stream or 0))
        if rc:
            self._h = C.c_void_p()
            raise BioEMError(rc, "bioem_create failed (no CUDA device? this library has no CPU fallback)")
        self.n_pix = 0
        self.n_models = 0
        self.n_img = 0
        self.max_shift = 0

    def _ck(self, rc):
        if rc:
            raise BioEMError(rc, self._L.bioem_last_error(self._h).decode())

    def close(self):
        if self._h:
            self._L.bioem_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def set_image_geometry(self, n_pix, pixel_size_A):
        self._ck(self._L.bioem_set_image_geometry(self._h, int(n_pix), float(pixel_size_A)))
        self.n_pix, self.n_img = int(n_pix), 0

    def clear_models(self):
        self._ck(self._L.bioem_clear_models(self._h))
        self.n_models = 0

    def add_model_atoms(self, xyz_A, radius_A, weight):
        xyz, xp = _f32(xyz_A)
        rad, rp = _f32(radius_A)
        wt, wp = _f32(weight)
        mid = C.c_int(-1)
        self._ck(self._L.bioem_add_model_atoms(self._h, len(rad), xp, rp, wp, C.byref(mid)))
        self.n_models += 1
        return mid.value

    def add_model_density(self, rho, voxel_A):
        rho, p = _f32(rho)
        mid = C.c_int(-1)
        self._ck(self._L.bioem_add_model_density(self._h, rho.shape[0], float(voxel_A), p, C.byref(mid)))
        self.n_models += 1
        return mid.value

    def set_orientations_quat(self, q_wxyz, log_prior=None):
        q, qp = _f32(q_wxyz)
        lp, lpp = (None, None) if log_prior is None else _f32(log_prior)
        self._ck(self._L.bioem_set_orientations_quat(self._h, len(q), qp, lpp))
        self.n_orient = len(q)

    def set_ctf_grid(self, a_A2, A, b_A2, log_prior=None):
        a, ap = _f32(a_A2)
        A_, Ap = _f32(A)
        b, bp = _f32(b_A2)
        lp, lpp = (None, None) if log_prior is None else _f32(log_prior)
        self._ck(self._L.bioem_set_ctf_grid(self._h, len(a), ap, Ap, bp, lpp))
        self.n_ctf = len(a)

    def set_shift_range(self, max_shift_px):
        self._ck(self._L.bioem_set_shift_range(self._h, int(max_shift_px)))
        self.max_shift = int(max_shift_px)

    def push_images(self, pixels):
        """pixels: float32 [n][N][N]; a numpy array (host) or a CUDA torch tensor (device, zero-copy)."""
        if hasattr(pixels, "data_ptr"):                       # torch tensor
            t = pixels.contiguous()
            if str(t.dtype) != "torch.float32":
                raise TypeError("push_images: float32 required")
            n = t.shape[0]
            self._ck(self._L.bioem_push_images(self._h, n, C.c_void_p(t.data_ptr()), 1 if t.is_cuda else 0))
        else:
            a, _ = _f32(pixels)
            n = a.shape[0]
            self._ck(self._L.bioem_push_images(self._h, n, C.c_void_p(a.ctypes.data), 0))
        self.n_img = n

    def run(self):
        self._ck(self._L.bioem_run(self._h))

    def invalidate_precompute(self):
        self._ck(self._L.bioem_invalidate_precompute(self._h))

    # ---- the run in phases (orientation sharding, include/bioem.h)
    def set_orientation_slice(self, o_begin=0, o_end=-1):
        self._ck(self._L.bioem_set_orientation_slice(self._h, int(o_begin), int(o_end)))
        self._slice = (int(o_begin), int(o_end)) if o_end >= 0 else None

    def run_partial(self):
        self._ck(self._L.bioem_run_partial(self._h))

    def get_partials_size(self):
        """(bytes of this context's partial blob, chunks per model in it)"""
        nb, nc = C.c_int64(), C.c_int32()
        self._ck(self._L.bioem_get_partials_size(self._h, C.byref(nb), C.byref(nc)))
        return nb.value, nc.value

    @staticmethod
    def _buf(t):
        """(address, is_device) of a contiguous torch tensor or numpy array"""
        if hasattr(t, "data_ptr"):
            assert t.is_contiguous()
            return C.c_void_p(t.data_ptr()), 1 if t.is_cuda else 0
        assert t.flags["C_CONTIGUOUS"]
        return C.c_void_p(t.ctypes.data), 0

    def export_partials(self, dst):
        p, dev = self._buf(dst)
        self._ck(self._L.bioem_export_partials(self._h, p, dev))

    def merge_partials(self, blobs=None, stride_bytes=0, chunks_of_blob=None):
        if blobs is None:
            self._ck(self._L.bioem_merge_partials(self._h, 0, None, 0, None, 1))
            return
        ch = np.ascontiguousarray(chunks_of_blob, dtype=np.int32)
        p, dev = self._buf(blobs)
        self._ck(self._L.bioem_merge_partials(self._h, len(ch), p, int(stride_bytes), ch.ctypes.data_as(_ip), dev))

    def rescore_local(self):
        self._ck(self._L.bioem_rescore_local(self._h))

    def rescore_shape(self):
        return (self.n_img, self.n_models, TOPK)

    def export_rescore(self, dst):
        p, dev = self._buf(dst)
        self._ck(self._L.bioem_export_rescore(self._h, p, dev))

    def import_rescore(self, src):
        p, dev = self._buf(src)
        self._ck(self._L.bioem_import_rescore(self._h, p, dev))

    def finish(self):
        self._ck(self._L.bioem_finish(self._h))

    def get_log_posterior(self):
        out = np.empty((self.n_img, self.n_models))
        self._ck(self._L.bioem_get_log_posterior(self._h, out.ctypes.data_as(_dp)))
        return out

    def get_best(self):
        shp = (self.n_img, self.n_models)
        o, c, dx, dy = (np.empty(shp, dtype=np.int32) for _ in range(4))
        lp = np.empty(shp)
        self._ck(self._L.bioem_get_best(self._h, o.ctypes.data_as(_ip), c.ctypes.data_as(_ip), dx.ctypes.data_as(_ip),
                                        dy.ctypes.data_as(_ip), lp.ctypes.data_as(_dp)))
        return dict(orient=o, ctf=c, dx=dx, dy=dy, log_p=lp)

    def set_displacement_variant(self, variant=0):
        """0 Fourier space / circular (default), 1 real space / cropping; before push_images."""
        self._ck(self._L.bioem_set_displacement_variant(self._h, int(variant)))

    def set_orientation_chunk(self, n_orient_per_item=0):
        self._ck(self._L.bioem_set_orientation_chunk(self._h, int(n_orient_per_item)))

    def debug_set_kernel(self, which=KERNEL_AUTO):
        self._ck(self._L.bioem_debug_set_kernel(self._h, int(which)))

    def get_run_plan(self):
        """(kernel, orientations per work item) of the last run."""
        k, oc = C.c_int(), C.c_int()
        self._ck(self._L.bioem_get_run_plan(self._h, C.byref(k), C.byref(oc)))
        return k.value, oc.value

    def get_run_plan_partial(self):
        """(kernel, orientations per work item) after run_partial (bioem_get_run_plan needs a finished run)."""
        k, oc = C.c_int(), C.c_int()
        self._ck(self._L.bioem_get_run_plan(self._h, C.byref(k), C.byref(oc)))
        return k.value, oc.value

    def set_orientation_posterior(self, enable=True):
        self._ck(self._L.bioem_set_orientation_posterior(self._h, int(bool(enable))))

    def get_orientation_log_posterior(self):
        """[n_img][n_model][orientations of this context's slice (the whole grid without one)]"""
        sl = getattr(self, "_slice", None)
        out = np.empty((self.n_img, self.n_models, sl[1] - sl[0] if sl else self.n_orient))
        self._ck(self._L.bioem_get_orientation_log_posterior(self._h, out.ctypes.data_as(_dp)))
        return out

    def get_ensemble_log_posterior(self, weights=None):
        """Eq. 10: (total, per_image)."""
        tot, per = np.empty(1), np.empty(self.n_img)
        wp = None
        if weights is not None:
            w = np.ascontiguousarray(weights, dtype=np.float64)
            assert w.shape == (self.n_models,)
            wp = w.ctypes.data_as(_dp)
        self._ck(self._L.bioem_get_ensemble_log_posterior(self._h, wp, tot.ctypes.data_as(_dp), per.ctypes.data_as(_dp)))
        return float(tot[0]), per

    @staticmethod
    def noalloc_last_error():
        return (lib().bioem_noalloc_last_error() or b"").decode()

    @staticmethod
    def noalloc_prepare(device=0):
        rc = lib().bioem_noalloc_prepare(device)
        if rc:
            raise BioEMError(rc, BioEM.noalloc_last_error())

    @staticmethod
    def ensemble_log_posterior_noalloc(log_p, weights, out_total, out_per_image=None, device=0, stream=0):
        """Eq. 10 without any allocation.  Every array is a CUDA float64 tensor (anything with data_ptr()) on `device`:
        log_p [n_img][n_model], weights [n_model] or None, out_total [1], out_per_image [n_img] or None; `stream` is a
        cudaStream_t (0 = default).  Enqueues and returns; the outputs are ready when the stream reaches them."""
        n_img, n_model = int(log_p.shape[0]), int(log_p.shape[1])
        ptr = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
        rc = lib().bioem_ensemble_log_posterior_noalloc(device, C.c_void_p(stream or 0), n_img, n_model, ptr(log_p), ptr(weights),
                                                        ptr(out_total), ptr(out_per_image))
        if rc:
            raise BioEMError(rc, BioEM.noalloc_last_error())

    def get_synthetic_map(self, model, orient, ctf, dx=0, dy=0, fit_to_image=None):
        """I_cal of Eq. 7 for one parameter set: (map [N][N] float32, normalisation N, offset mu)."""
        out = np.empty((self.n_pix, self.n_pix), dtype=np.float32)
        no = np.zeros(2)
        fp = None
        if fit_to_image is not None:
            img, fp = _f32(fit_to_image)
            assert img.shape == (self.n_pix, self.n_pix)
        self._ck(self._L.bioem_get_synthetic_map(self._h, model, orient, ctf, int(dx), int(dy), fp, out.ctypes.data_as(_fp), no.ctypes.data_as(_dp)))
        return out, float(no[0]), float(no[1])

    def debug_calc_image(self, model, orient, ctf):
        out = np.empty((self.n_pix, self.n_pix), dtype=np.float32)
        self._ck(self._L.bioem_debug_calc_image(self._h, model, orient, ctf, out.ctypes.data_as(_fp)))
        return out

    def debug_shift_map(self, img, model, orient, ctf, f64=False):
        S1 = 2 * self.max_shift + 1
        out = np.empty((S1, S1))
        fn = self._L.bioem_debug_shift_map_f64 if f64 else self._L.bioem_debug_shift_map
        self._ck(fn(self._h, img, model, orient, ctf, out.ctypes.data_as(_dp)))
        return out

    def debug_shift_map_f64(self, img, model, orient, ctf):
        return self.debug_shift_map(img, model, orient, ctf, f64=True)

    def debug_log_posterior_f32(self):
        out = np.empty((self.n_img, self.n_models))
        self._ck(self._L.bioem_debug_log_posterior_f32(self._h, out.ctypes.data_as(_dp)))
        return out

    def get_timing(self):
        a, b = C.c_double(), C.c_double()
        self._ck(self._L.bioem_get_timing(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def get_launch_count(self):
        a, b = C.c_int64(), C.c_int64()
        self._ck(self._L.bioem_get_launch_count(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def measure_fp32_peak(self):
        a, b = C.c_double(), C.c_double()
        self._ck(self._L.bioem_measure_fp32_peak(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    # convenience: load a bioem_workloads dict
    def load_workload(self, wl, images=True):
        s = wl["spec"]
        self.set_image_geometry(s.n_pix, s.pixel_A)
        self.clear_models()
        for m in wl["models"]:
            if m["kind"] == "atoms":
                self.add_model_atoms(m["xyz"], m["radius"], m["weight"])
            else:
                self.add_model_density(m["rho"], m["voxel_A"])
        self.set_orientations_quat(wl["quats"])
        self.set_ctf_grid(wl["ctfs"][:, 0], wl["ctfs"][:, 1], wl["ctfs"][:, 2])
        self.set_shift_range(s.max_shift)
        if images:
            self.push_images(wl["images"])
