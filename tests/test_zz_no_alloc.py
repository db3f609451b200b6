"""sph_cell_scan_static (include/sph.h): row a3's exclusive scan on a file-scope `static __device__` scratch array, for callers
that may not call cudaMalloc.  Its output is compared with the EXISTING path's -- the cell_start array the rebuild chain of a
context leaves behind (scan_cells with context-owned scratch), exported as SPH_FIELD_SORT_CELL_START from the histogram
SPH_FIELD_SORT_CELL_COUNT -- bit for bit (integer work: the bar of every index comparison in these tests), on several calls in
a row that share the scratch array.

The file is named so that pytest collects it last (`pytest --collect-only`): the suite runs with `pytest -x`, and a failure
here must not hide the other tests.  It passes alone in a fresh process (the first call resolves the scratch address) and after
the other tests.
"""
import numpy as np
import pytest

from paper_2512_09904_b200 import workloads as wl


@pytest.fixture(scope="module")
def api():
    from paper_2512_09904_b200 import api as _api
    _api.lib()                      # fails loudly if libsph_b200.so is missing
    return _api


def _existing_path(api, w, **over):
    """histogram and cell_start of the context's own rebuild (the existing path, scratch in context memory)."""
    sim = api.Simulation(w, **over)
    sim.step(1)
    sim.sync()
    st = sim.stats()
    n_cells = 4 * int(st["ncell_x"]) * int(st["ncell_y"]) * int(st["ncell_z"])
    counts, starts = sim.get("SORT_CELL_COUNT").copy(), sim.get("SORT_CELL_START").copy()
    sim.close()
    assert counts.shape == (n_cells,) and starts.shape == (n_cells + 1,)
    assert int(counts.sum(dtype=np.uint64)) == w.n_f == int(starts[-1])
    return counts, starts


def _scan_static(api, torch, counts, n_items, poison, check_mem=True):
    """one call of the new entry point on caller-owned device buffers; returns the host copy of starts."""
    n = len(counts)
    c = torch.from_numpy(counts.view(np.int32)).cuda()
    s = torch.full((n + 1,), poison, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    api.sph_cell_scan_static(0, c, s, n, n_items, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    # (not on a process's first call: resolving the scratch address may make the driver load the library's device code)
    assert not check_mem or torch.cuda.mem_get_info()[0] == free0, "the call changed the device's free memory"
    assert np.array_equal(c.cpu().numpy().view(np.uint32), counts), "the input was modified"
    return s.cpu().numpy().view(np.uint32)


@pytest.mark.gpu
def test_static_scan_matches_the_rebuild_chain_on_calls_in_a_row(api):
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    over = dict(dt_fixed=2e-5, rebuild_every=1)
    small = _existing_path(api, wl.perturb_state(wl.still_tank(n=16)), **over)                   # 2 scan blocks
    big = _existing_path(api, wl.random_cloud(60000, 20000, extent=(40, 30, 20), seed=5), **over)  # > 20 blocks
    assert len(big[0]) > 20 * 2048 > len(small[0])
    # calls in a row on the shared scratch: small, big, small again (stale partial sums of the bigger call behind it), big
    for k, (counts, starts) in enumerate((small, big, small, big)):
        got = _scan_static(api, torch, counts, int(starts[-1]), poison=0x5a5a5a5a if k % 2 else -1, check_mem=k > 0)
        assert np.array_equal(got, starts), f"call {k}: {np.flatnonzero(got != starts)[:5]}"
        want = np.concatenate(([0], np.cumsum(counts, dtype=np.uint64))).astype(np.uint32)       # the definition, as a cross-check
        want[-1] = starts[-1]
        assert np.array_equal(got, want)


@pytest.mark.gpu
def test_static_scan_at_many_blocks_and_at_the_edges(api):
    """more than 256 scan blocks (k_scan_sums walks its partial sums in several rounds), one cell, exact multiples of a block."""
    import torch
    rng = np.random.default_rng(11)
    for n in (1, 2047, 2048, 2049, 256 * 2048, 256 * 2048 + 1, 3_000_001):
        counts = rng.integers(0, 40, size=n, dtype=np.uint32)
        got = _scan_static(api, torch, counts, 123456789, poison=-1, check_mem=n > 1)
        want = np.concatenate(([0], np.cumsum(counts, dtype=np.uint64))).astype(np.uint32)
        want[-1] = 123456789                                                                      # starts[n_cells] = n_items as passed
        assert np.array_equal(got, want), n


def test_static_scan_rejects_sizes_beyond_its_scratch(api):
    """no GPU needed: the checks come before any CUDA call."""
    for n_cells in (0, api.SCAN_STATIC_MAX_CELLS + 1):
        with pytest.raises(api.SphError) as e:
            api.sph_cell_scan_static(0, 0x1000, 0x100000000, n_cells, 0)
        assert e.value.code == api.SPH_EINVAL and "SPH_SCAN_STATIC_MAX_CELLS" in str(e.value)
    with pytest.raises(api.SphError) as e:
        api.sph_cell_scan_static(0, 0, 0x1000, 16, 0)
    assert "NULL" in str(e.value)
    with pytest.raises(api.SphError) as e:
        api.sph_cell_scan_static(0, 0x1000, 0x1020, 16, 0)
    assert "overlap" in str(e.value)
