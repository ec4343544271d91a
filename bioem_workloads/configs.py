"""The five BASELINE.json configs plus reduced "mini" variants of each for
element-by-element parity in seconds.  Pure data: no arithmetic of the method lives here."""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Tuple

BASE_SEED = 160906634  # arXiv id of the paper; + config index


@dataclass(frozen=True)
class WorkloadSpec:
    name: str
    index: int                      # position in BASELINE.json "configs"
    n_pix: int                      # N (square images)
    pixel_A: float
    max_shift: int                  # D; shifts are all integer |dx|,|dy| <= D (R6)
    n_images: int
    model: str                      # "atoms" | "density" | "ensemble"
    n_atoms: int = 0
    ball_A: float = 0.0
    radius_A: Tuple[float, float] = (1.5, 1.5)     # uniform range
    weight: Tuple[float, float] = (1.0, 1.0)
    n_models: int = 1
    n_source_models: int = 1        # ensemble: how many of the models generate images
    orient_grid: str = "euler"      # "euler" (n^3 mid-point ZYZ grid) | "hopf" (Fibonacci S2 x psi)
    orient_shape: Tuple[int, ...] = (4, 4, 4)
    orient_stride: int = 1          # mini variants keep every k-th grid orientation
    defocus_um: Tuple[float, ...] = (1.0, 2.0)
    bfactor_A2: Tuple[float, ...] = (0.0, 50.0)
    amp_contrast: Tuple[float, ...] = (0.1,)
    snr: Tuple[float, float] = (0.1, 0.1)
    kV: float = 300.0
    # density model
    n_vox: int = 0
    n_blobs: int = 0
    blob_sigma_A: float = 2.0

    @property
    def seed(self) -> int:
        return BASE_SEED + self.index

    @property
    def n_orient(self) -> int:
        n = 1
        for s in self.orient_shape:
            n *= s
        return len(range(0, n, self.orient_stride))

    @property
    def n_ctf(self) -> int:
        return len(self.defocus_um) * len(self.bfactor_A2) * len(self.amp_contrast)

    @property
    def n_shifts(self) -> int:
        return (2 * self.max_shift + 1) ** 2

    @property
    def n_pairs(self) -> int:
        return self.n_images * self.n_models * self.n_orient * self.n_ctf

    @property
    def n_evaluations(self) -> int:
        return self.n_pairs * self.n_shifts


def _lin(a, b, n):
    return tuple(a + (b - a) * i / (n - 1) for i in range(n))


_TINY = WorkloadSpec(
    name="tiny", index=0, n_pix=64, pixel_A=2.0, max_shift=4, n_images=16, model="atoms", n_atoms=200,
    ball_A=30.0, orient_grid="euler", orient_shape=(4, 4, 4), defocus_um=(1.0, 2.0), bfactor_A2=(0.0, 50.0),
    amp_contrast=(0.1,), snr=(0.1, 0.1))

_SMALL = WorkloadSpec(
    name="small", index=1, n_pix=128, pixel_A=1.5, max_shift=16, n_images=256, model="atoms", n_atoms=2000,
    ball_A=50.0, orient_grid="hopf", orient_shape=(192, 24), defocus_um=_lin(0.5, 3.0, 4),
    bfactor_A2=(0.0, 50.0, 100.0, 150.0), amp_contrast=(0.05, 0.1), snr=(0.1, 0.1))

_PAPER = WorkloadSpec(
    name="paper", index=2, n_pix=224, pixel_A=1.0, max_shift=30, n_images=1024, model="atoms", n_atoms=10000,
    ball_A=70.0, radius_A=(1.0, 2.0), weight=(1.0, 8.0), orient_grid="euler", orient_shape=(16, 16, 16),
    defocus_um=_lin(0.5, 3.0, 8), bfactor_A2=(0.0, 50.0, 100.0, 150.0), amp_contrast=(0.1,), snr=(0.05, 0.2))

_DENSITY = WorkloadSpec(
    name="density", index=3, n_pix=128, pixel_A=1.5, max_shift=12, n_images=2048, model="density", n_vox=128,
    n_blobs=5000, ball_A=50.0, blob_sigma_A=2.0, orient_grid="hopf", orient_shape=(384, 24),
    defocus_um=_lin(0.5, 3.0, 4), bfactor_A2=(0.0, 50.0, 100.0, 150.0), amp_contrast=(0.1,), snr=(0.1, 0.1))

_ENSEMBLE = WorkloadSpec(
    name="ensemble", index=4, n_pix=128, pixel_A=1.5, max_shift=10, n_images=512, model="ensemble", n_atoms=3000,
    ball_A=40.0, n_models=64, n_source_models=4, orient_grid="hopf", orient_shape=(96, 12),
    defocus_um=_lin(0.5, 3.0, 4), bfactor_A2=(0.0, 100.0), amp_contrast=(0.1,), snr=(0.1, 0.1))

CONFIGS = {s.name: s for s in (_TINY, _SMALL, _PAPER, _DENSITY, _ENSEMBLE)}

# Reduced variants: same recipe, same image size / shift range / model, fewer images, a strided subset of the
# orientation grid and a sub-grid of CTFs -- small enough for the direct-summation oracle to finish in seconds,
# large enough to span several CTAs / tiles and a ragged tail (odd counts on purpose).
CONFIGS["small_mini"] = replace(_SMALL, name="small_mini", n_images=7, orient_stride=921,
                                defocus_um=(0.5, 3.0), bfactor_A2=(0.0, 150.0), amp_contrast=(0.1,))
CONFIGS["paper_mini"] = replace(_PAPER, name="paper_mini", n_images=3, orient_stride=1365,
                                defocus_um=(0.5, 3.0), bfactor_A2=(50.0,))
CONFIGS["density_mini"] = replace(_DENSITY, name="density_mini", n_images=9, orient_stride=1843,
                                  defocus_um=(0.5, 3.0), bfactor_A2=(0.0, 150.0))
CONFIGS["ensemble_mini"] = replace(_ENSEMBLE, name="ensemble_mini", n_images=6, n_models=3, n_source_models=2,
                                   orient_stride=230, defocus_um=(0.5, 3.0), bfactor_A2=(100.0,))
CONFIGS["tiny_mini"] = replace(_TINY, name="tiny_mini", n_images=5, orient_stride=13)


# "mid" variants: >= 40 orientations and >= 7 CTFs (three CTF groups of the packed kernel, an orientation change in the middle
# of a work item's software pipeline), still seconds for the direct-summation oracle: the element-by-element parity cases of
# the chunked launch (orientations per work item 1, 2, 5, 32).
CONFIGS["tiny_mid"] = replace(_TINY, name="tiny_mid", n_images=6, defocus_um=(1.0, 1.5, 2.0, 2.5))
CONFIGS["small_mid"] = replace(_SMALL, name="small_mid", n_images=5, orient_stride=107,
                               bfactor_A2=(0.0, 150.0), amp_contrast=(0.1,))
CONFIGS["paper_mid"] = replace(_PAPER, name="paper_mid", n_images=3, orient_stride=97,
                               defocus_um=_lin(0.5, 3.0, 7), bfactor_A2=(50.0,))
CONFIGS["ensemble_mid"] = replace(_ENSEMBLE, name="ensemble_mid", n_images=4, n_models=3, n_source_models=2,
                                  orient_stride=28, defocus_um=_lin(0.5, 3.0, 4), bfactor_A2=(0.0, 100.0))


# Other box sizes: 170^2 is the GroEL set of the paper's Table 1, 2 x 5 x 17: no power-of-two factor beyond 2.
# Same recipe as Small (2,000 atoms, 1.5 A/px), shift range +-6, a handful of images / orientations / CTFs: parity cases only.
for _n in (96, 160, 170, 192):
    CONFIGS[f"box{_n}_mini"] = replace(_SMALL, name=f"box{_n}_mini", n_pix=_n, max_shift=6, n_images=4, orient_stride=1151,
                                       defocus_um=(0.5, 3.0), bfactor_A2=(50.0,), amp_contrast=(0.1,))


def get_spec(name: str, **overrides) -> WorkloadSpec:
    spec = CONFIGS[name]
    return replace(spec, **overrides) if overrides else spec
