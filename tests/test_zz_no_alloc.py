"""The allocation-free entry point (include/bioem.h, bioem_ensemble_log_posterior_noalloc; csrc/noalloc.cu) against the
existing, allocating path (bioem_get_ensemble_log_posterior) on the same log-posteriors: two calls in a row through the shared
file-scope work array, the size limit, and that device memory in use does not move.  Collected last on purpose (the name):
the suite runs with pytest -x."""
import numpy as np
import pytest

import bioem_workloads as W

pytestmark = pytest.mark.gpu

# Both sides are FP64 with the same summation order; they differ only in log() of the weights (host libm there, device here).
RTOL = 1e-12


def _existing_path(name, weight_sets):
    from paper_1609_06634_b200 import BioEM
    wl = W.build_workload(name)
    with BioEM() as b:
        b.load_workload(wl)
        b.run()
        logp = b.get_log_posterior()
        want = [b.get_ensemble_log_posterior(w) for w in weight_sets]
    return logp, want


def test_noalloc_ensemble_matches_existing_path_twice_in_a_row():
    import torch
    from paper_1609_06634_b200 import BioEM
    w = np.array([0.5, 0.3, 0.2])
    weight_sets = [None, w, np.array([1.0, 0.0, 0.0])]
    logp, want = _existing_path("ensemble_mini", weight_sets)
    n_img, n_model = logp.shape
    assert n_model == 3 and n_img >= 2
    dev = torch.device("cuda", 0)
    d_logp = torch.from_numpy(logp).to(dev)
    d_w = [None if x is None else torch.from_numpy(x).to(dev) for x in weight_sets]
    d_tot = torch.full((len(weight_sets),), float("nan"), dtype=torch.float64, device=dev)
    d_per = torch.full((len(weight_sets), n_img), float("nan"), dtype=torch.float64, device=dev)
    stream = torch.cuda.current_stream(dev).cuda_stream
    BioEM.noalloc_prepare(0)
    # warm call (loads the two kernels), then the calls that are checked: back to back on one stream, no sync in between
    BioEM.ensemble_log_posterior_noalloc(d_logp, None, d_tot[0:1], d_per[0], device=0, stream=stream)
    torch.cuda.synchronize()
    free_before = None
    for rep in range(3):
        if rep == 1:                                                  # everything below has run once: torch's kernels are loaded too
            free_before, _ = torch.cuda.mem_get_info(dev)
        d_tot.fill_(float("nan"))
        d_per.fill_(float("nan"))
        for k in range(len(weight_sets)):
            BioEM.ensemble_log_posterior_noalloc(d_logp, d_w[k], d_tot[k:k + 1], d_per[k], device=0, stream=stream)
        torch.cuda.synchronize()
        tot, per = d_tot.cpu().numpy(), d_per.cpu().numpy()
        for k, (rtot, rper) in enumerate(want):
            assert abs(tot[k] - rtot) <= RTOL * abs(rtot), (rep, k, tot[k], rtot)
            assert np.abs(per[k] - rper).max() <= RTOL * np.abs(rper).max(), (rep, k)
    free_after, _ = torch.cuda.mem_get_info(dev)
    assert free_after >= free_before, (free_before, free_after)      # nothing was allocated on the device by the last six calls


def test_noalloc_stale_contents_and_optional_output():
    """The work array keeps the last call's entries: a call on fewer images after a call on more must not see them."""
    import torch
    from paper_1609_06634_b200 import BioEM
    logp, want = _existing_path("ensemble_mini", [None])
    n_img = logp.shape[0]
    dev = torch.device("cuda", 0)
    d_logp = torch.from_numpy(logp).to(dev)
    big = torch.from_numpy(np.tile(logp, (5, 1)) + 7.0).to(dev)       # more images, different values, left in the array
    d_tot = torch.zeros(2, dtype=torch.float64, device=dev)
    BioEM.ensemble_log_posterior_noalloc(big, None, d_tot[0:1], None)
    BioEM.ensemble_log_posterior_noalloc(d_logp, None, d_tot[1:2], None)                 # out_per_image = NULL
    torch.cuda.synchronize()
    tot = d_tot.cpu().numpy()
    rtot = want[0][0]
    assert abs(tot[1] - rtot) <= RTOL * abs(rtot)
    # the large call: 5 copies shifted by 7 in the log.  Different summation order from 5 * (rtot + 7 n_img), so looser.
    assert abs(tot[0] - 5 * (rtot + 7.0 * n_img)) <= 1e-9 * abs(tot[0])


def test_noalloc_rejects_sizes_beyond_the_work_array():
    import torch
    from paper_1609_06634_b200 import BioEM, BioEMError
    from paper_1609_06634_b200 import binding
    dev = torch.device("cuda", 0)
    out = torch.full((1,), 123.0, dtype=torch.float64, device=dev)
    too_many = torch.zeros((binding.NOALLOC_MAX_IMG + 1, 1), dtype=torch.float64, device=dev)
    with pytest.raises(BioEMError) as e:
        BioEM.ensemble_log_posterior_noalloc(too_many, None, out)
    assert e.value.code == -5 and "at most" in str(e.value)
    too_wide = torch.zeros((2, binding.NOALLOC_MAX_MODEL + 1), dtype=torch.float64, device=dev)
    with pytest.raises(BioEMError) as e:
        BioEM.ensemble_log_posterior_noalloc(too_wide, None, out)
    assert e.value.code == -5
    torch.cuda.synchronize()
    assert out.item() == 123.0                                        # nothing was enqueued
    # the largest accepted size runs: all log P = 0, uniform weights -> every inner sum is log(1) = 0
    full = torch.zeros((binding.NOALLOC_MAX_IMG, 2), dtype=torch.float64, device=dev)
    per = torch.full((binding.NOALLOC_MAX_IMG,), float("nan"), dtype=torch.float64, device=dev)
    BioEM.ensemble_log_posterior_noalloc(full, None, out, per)
    torch.cuda.synchronize()
    assert abs(out.item()) <= 1e-9 and per.abs().max().item() <= 1e-15


def test_noalloc_entry_point_under_graph_capture():
    """What the entry point is for: it can be captured into a CUDA graph (nothing in it allocates or synchronises) and replayed on
    new contents of the same buffers."""
    import torch
    from paper_1609_06634_b200 import BioEM
    dev = torch.device("cuda", 0)
    rng = np.random.default_rng(0)
    logp = torch.from_numpy(rng.normal(size=(1000, 5)) * 10 - 3000).to(dev)
    w = torch.tensor([0.1, 0.2, 0.3, 0.25, 0.15], dtype=torch.float64, device=dev)
    tot = torch.zeros(1, dtype=torch.float64, device=dev)
    per = torch.zeros(1000, dtype=torch.float64, device=dev)
    BioEM.noalloc_prepare(0)                                         # the symbol's address is taken before the capture begins
    BioEM.ensemble_log_posterior_noalloc(logp, w, tot, per)          # eager: loads the kernels, gives the expected values
    torch.cuda.synchronize()
    want_tot, want_per = tot.item(), per.clone()
    tot.zero_(); per.zero_()
    torch.cuda.synchronize()
    graph, side = torch.cuda.CUDAGraph(), torch.cuda.Stream()
    with torch.cuda.graph(graph, stream=side):
        BioEM.ensemble_log_posterior_noalloc(logp, w, tot, per, device=0, stream=torch.cuda.current_stream().cuda_stream)
    assert tot.item() == 0.0                                         # captured, not run
    graph.replay()
    torch.cuda.synchronize()
    assert tot.item() == want_tot and torch.equal(per, want_per)
    logp += 1.0                                                      # every log P up by one: every inner sum too
    graph.replay()
    torch.cuda.synchronize()
    assert abs(tot.item() - (want_tot + 1000.0)) <= 1e-9 * abs(want_tot) and (per - want_per - 1.0).abs().max().item() <= 1e-9
