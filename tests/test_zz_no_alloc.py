"""cpm_update_statistics_noalloc (include/cpm.h): the update-statistics kernel on the library's file-scope
`static __device__` scratch array, for callers that cannot call cudaMalloc.  Its output must equal
cpm_update_statistics bit for bit (integer histograms: the bar of the other GPU tests), on two calls in a row --
the array keeps the previous call's contents -- and sizes beyond the stated maximum are refused.

Collected last on purpose (pytest -x): a failure here hides nothing."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pk():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2312_09317_b200 as m
    m.load_library()
    return m


def _ctx(pk, name, dims, **over):
    import cpm_inputs as ci
    cfg = ci.make_config(name, dims=dims)
    p = dict(cfg["params"]); p.update(over)
    g = pk.CPM(cfg["dims"], max_cells=cfg["max_cells"], **p)
    g.set_lattice(cfg["ids"], cfg["frozen"], cfg["cell_type"])
    return g


def test_noalloc_statistics_equal_existing_path_twice_in_a_row(pk):
    """Two different contexts back to back on the shared array (2D then 3D, the second smaller than the first so
    stale words of the first call lie beyond and inside its range), host outputs; then the first again with other
    histogram sizes.  Every result equals cpm_update_statistics."""
    pk.noalloc_setup(0)
    a = _ctx(pk, "C1", (64, 48), subsection=8, attempts_per_activation=16)
    b = _ctx(pk, "C2", (16, 16, 16), subsection=4, attempts_per_activation=64)
    a.step(3); b.step(2)
    for g, n_mcs, nf, nw, wb in ((a, 20, 8, 200, 4), (b, 20, 8, 200, 4), (a, 7, 5, 64, 1), (b, 12, 16, 33, 9)):
        f_ref, w_ref = g.update_statistics(n_mcs, n_freq=nf, n_wait=nw, wait_bin=wb)
        for _ in range(2):
            f = np.full(nf, 0xDEAD, np.uint64); w = np.full(nw, 0xBEEF, np.uint64)
            g.update_statistics_noalloc(n_mcs, f, w, wait_bin=wb)
            np.testing.assert_array_equal(f, f_ref)
            np.testing.assert_array_equal(w, w_ref)
        assert int(f_ref.sum()) == (64 * 48 if g is a else 16 ** 3) * n_mcs


def test_noalloc_statistics_device_outputs(pk):
    """Caller-owned DEVICE outputs: results in stream order, equal to the existing path, twice in a row."""
    import torch
    g = _ctx(pk, "C1", (128, 128), subsection=8)
    g.step(2)
    f_ref, w_ref = g.update_statistics(10, n_freq=8, n_wait=128, wait_bin=2)
    f = torch.empty(8, dtype=torch.int64, device="cuda:0"); w = torch.empty(128, dtype=torch.int64, device="cuda:0")
    for _ in range(2):
        f.fill_(-1); w.fill_(-1)
        torch.cuda.synchronize()
        g.update_statistics_noalloc(10, f, w, wait_bin=2)
        torch.cuda.synchronize()
        np.testing.assert_array_equal(f.cpu().numpy().view(np.uint64), f_ref)
        np.testing.assert_array_equal(w.cpu().numpy().view(np.uint64), w_ref)
    # the state is untouched: the run goes on as a context that never asked
    h = _ctx(pk, "C1", (128, 128), subsection=8)
    h.step(3); g.step(1)
    np.testing.assert_array_equal(g.get_lattice(), h.get_lattice())


def test_noalloc_statistics_allocates_no_device_memory(pk):
    """Free device memory does not shrink over the calls (the array was placed when the library loaded)."""
    import torch
    g = _ctx(pk, "C1", (256, 256), subsection=8)
    f = np.zeros(8, np.uint64); w = np.zeros(64, np.uint64)
    g.update_statistics_noalloc(2, f, w)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info(0)[0]
    for _ in range(3):
        g.update_statistics_noalloc(2, f, w)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info(0)[0] >= free0   # nothing was taken (a context of an earlier test freed in between may add)


def test_noalloc_statistics_refuses_sizes_beyond_the_maximum(pk):
    """More than CPM_NOALLOC_MAX_SITES sites, or more than CPM_NOALLOC_MAX_BINS bins: CPM_ERR_ARG naming the limit;
    the largest lattice that fits is served."""
    assert pk.NOALLOC_MAX_SITES == 1 << 20 and pk.NOALLOC_MAX_BINS == 4096
    big = _ctx(pk, "C1", (1024, 1032), subsection=8)
    f = np.zeros(8, np.uint64); w = np.zeros(64, np.uint64)
    with pytest.raises(pk.CPMError) as ei:
        big.update_statistics_noalloc(1, f, w)
    assert "CPM_NOALLOC_MAX_SITES" in str(ei.value)
    f_ref, _ = big.update_statistics(1, n_freq=8, n_wait=64)      # the allocating path still serves it
    assert int(f_ref.sum()) == 1024 * 1032
    edge = _ctx(pk, "C1", (1024, 1024), subsection=8)
    edge.update_statistics_noalloc(1, f, w)
    f_ref, w_ref = edge.update_statistics(1, n_freq=8, n_wait=64)
    np.testing.assert_array_equal(f, f_ref)
    np.testing.assert_array_equal(w, w_ref)
    with pytest.raises(pk.CPMError):
        edge.update_statistics_noalloc(1, np.zeros(4000, np.uint64), np.zeros(97, np.uint64))
