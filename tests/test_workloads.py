"""The synthetic microscope renders the same forward model as the oracle (so planted parameters are the
best-scoring ones), and the grids are duplicate-free (R15).  CPU only."""
import numpy as np

import oracle
import bioem_workloads as W
from bioem_workloads import simulate


def test_atom_renderer_matches_oracle_forward_model():
    wl = W.build_workload("tiny_mini", with_images=False)
    s = wl["spec"]
    for o, c in ((0, 0), (3, 2)):
        a = oracle.calc_image(wl["models"][0], wl["quats"][o], wl["ctfs"][c], s.n_pix, s.pixel_A)
        b = simulate.render_signal(wl["models"][0], wl["quats"][o], wl["ctfs"][c], s.n_pix, s.pixel_A)
        assert np.abs(a - b).max() < 1e-11 * np.abs(a).max()


def test_density_renderer_matches_oracle_forward_model():
    spec = W.get_spec("density_mini", n_vox=32, n_pix=32, n_blobs=40, ball_A=14.0)
    model = W.make_density_model(spec)
    quats = W.generate.orientation_grid(spec)
    ctf = W.ctf_grid(spec)[1]
    om = oracle.prepare_model(model)
    for q in quats[:3]:
        a = oracle.calc_image(om, q, ctf, 32, spec.pixel_A)
        b = simulate.render_signal(model, q, ctf, 32, spec.pixel_A)
        assert np.abs(a - b).max() < 1e-9 * np.abs(a).max()


def test_grids_are_duplicate_free_and_sized():
    for name, want in (("tiny", 64), ("small", 4608), ("paper", 4096), ("density", 9216), ("ensemble", 1152)):
        spec = W.get_spec(name)
        q = W.generate.orientation_grid(spec)
        assert q.shape == (want, 4) and spec.n_orient == want
        assert np.allclose(np.linalg.norm(q, axis=1), 1.0)
        if want <= 4608:
            # q and -q are the same rotation: canonicalise the sign, then look for near-duplicates
            qc = q * np.where(q[:, :1] < 0, -1.0, 1.0)
            g = np.abs(qc @ qc.T)
            np.fill_diagonal(g, 0.0)
            assert g.max() < 1 - 1e-6
    assert [W.get_spec(n).n_ctf for n in ("tiny", "small", "paper", "density", "ensemble")] == [4, 32, 32, 16, 8]
    assert W.get_spec("small").n_evaluations == 256 * 4608 * 32 * 33 * 33
    assert W.get_spec("ensemble").n_pairs == 512 * 64 * 1152 * 8


def test_workload_is_seeded_and_float32():
    a = W.build_workload("tiny_mini")
    b = W.build_workload("tiny_mini")
    assert a["images"].dtype == np.float32 and np.array_equal(a["images"], b["images"])
    assert np.array_equal(a["quats"], b["quats"])


def test_ensemble_models_are_hinge_perturbations():
    spec = W.get_spec("ensemble_mini")
    models = W.make_ensemble_models(spec)
    base = W.make_atom_model(spec)
    assert len(models) == 3
    for m in models:
        moved = np.linalg.norm(m["xyz"] - base["xyz"], axis=1) > 1e-9
        assert 0.2 < moved.mean() < 0.8          # roughly one side of a plane through the centroid
        # rigid: pairwise distances inside the moved part are preserved
        a, b = m["xyz"][moved][:20], base["xyz"][moved][:20]
        assert np.allclose(np.linalg.norm(a[:, None] - a[None], axis=-1), np.linalg.norm(b[:, None] - b[None], axis=-1))


def test_bench_helpers():
    """bench.py's roofline inputs: the pruned flop count of SURVEY 8(d) / DESIGN 7 and the committed ncu table."""
    import importlib.util
    from pathlib import Path
    spec = importlib.util.spec_from_file_location("bench", Path(__file__).resolve().parent.parent / "bench.py")
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    # 6H + (N/2+1) 5 N log2 N + (2D+1) 2.5 N log2 N + 30 S, written out for Small and Paper-scale
    assert abs(bench.algorithmic_flops_per_pair(128, 16) - (6 * 8320 + 65 * 5 * 128 * 7 + 33 * 2.5 * 128 * 7 + 30 * 1089)) < 1e-6
    assert abs(bench.algorithmic_flops_per_pair(224, 30) - 1518300.083) < 1.0
    row = bench.ncu_table("paper")
    assert row is not None and row["kernel"] == "k_fused_tm" and float(row["dram_bytes_per_launch"]) > 1e9
    assert (Path(bench.ROOT) / row["capture"].split(" ")[0]).exists()              # the capture the row cites is committed
    assert bench.ncu_table("no such workload") is None
    assert W.get_spec("paper").n_evaluations == 1024 * 4096 * 32 * 61 * 61         # the bench default (config.workload)
