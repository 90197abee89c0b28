"""Host transfers of a large lattice go slab by slab, overlapped with the pack / recount / unpack kernels (cpm_lib.cu:
pipe_plan).  The slab arithmetic (odd numbers of subsection layers, periodic wrap of the first slab, groups that straddle
two slabs, both colour bits) is checked here on small lattices by lowering the size threshold through the environment
variable CPM_PIPE_MIN_SITES: the state after cpm_set_lattice, the read-back and a few MCS must equal the oracle's bit for
bit, exactly as on the one-piece path.  Needs a B200 (`-m gpu`)."""
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


CASES = [
    ("C4", (32, 24, 132), 4, (0, 0, 0)),     # 33 layers along z: the last pair of layers is half empty
    ("C4", (32, 32, 128), 4, (1, 1, 1)),     # periodic: slab 0 reads the last slab's top plane and goes last
    ("C2", (16, 16, 64), 2, (0, 0, 1)),
    ("C3", (64, 32, 136), 4, (1, 0, 0)),     # 34 layers = 17 pairs over 8 slabs: uneven slabs
    ("C5", (128, 264), 8, (0, 0, 0)),        # 2D: slabs along y, 33 layers
    ("C5", (64, 128), 4, (1, 1, 0)),
    ("C5", (256, 512), 16, (0, 1, 0)),
]


@pytest.mark.parametrize("name,dims,S,periodic", CASES)
def test_piped_transfers_equal_oracle(pk, oracle_mod, monkeypatch, name, dims, S, periodic):
    import cpm_inputs as ci
    cfg = ci.make_config(name, dims=dims)
    p = dict(cfg["params"]); p.update(subsection=S, periodic=periodic)
    monkeypatch.setenv("CPM_PIPE_MIN_SITES", str(1 << 40))
    whole = pk.CPM(cfg["dims"], max_cells=cfg["max_cells"], **p)
    monkeypatch.setenv("CPM_PIPE_MIN_SITES", "1")
    g = pk.CPM(cfg["dims"], max_cells=cfg["max_cells"], **p)
    o = oracle_mod.Oracle(cfg["dims"], max_cells=cfg["max_cells"], **p)
    for x in (whole, g, o):
        x.set_lattice(cfg["ids"], cfg["frozen"], cfg["cell_type"])
    assert g.get_launch_info()["pooled"]
    # the slab path really ran: it launches pack and recount once per slab and colour
    assert g.get_launch_info()["launches"] >= whole.get_launch_info()["launches"] + 6 * (1 << len(dims))
    for it in range(2):
        np.testing.assert_array_equal(g.get_lattice(), o.get_lattice())
        sg, so = g.get_cell_stats(), o.get_cell_stats()
        for k in so:
            np.testing.assert_array_equal(sg[k], so[k], err_msg="%s after %d MCS" % (k, 3 * it))
        g.step(3); o.step(3)
    whole.step(6)
    np.testing.assert_array_equal(g.get_lattice(), o.get_lattice())
    np.testing.assert_array_equal(g.get_lattice(), whole.get_lattice())
    # a second set_lattice on the same context (the staging buffers and events are reused)
    g.set_lattice(cfg["ids"], cfg["frozen"], cfg["cell_type"])
    g.set_mcs(0)
    g.step(6)
    np.testing.assert_array_equal(g.get_lattice(), whole.get_lattice())


def test_small_geometries_fall_back_to_one_piece(pk, oracle_mod, monkeypatch):
    """Fewer than 16 pairs of layers, or fewer than 8 chains per layer: no slabs, same result."""
    import cpm_inputs as ci
    monkeypatch.setenv("CPM_PIPE_MIN_SITES", "1")
    for name, dims, S in (("C4", (16, 16, 256), 8), ("C2", (32, 32, 32), 4), ("C5", (32, 512), 8)):
        cfg = ci.make_config(name, dims=dims)
        p = dict(cfg["params"]); p.update(subsection=S)
        g = pk.CPM(cfg["dims"], max_cells=cfg["max_cells"], **p)
        o = oracle_mod.Oracle(cfg["dims"], max_cells=cfg["max_cells"], **p)
        g.set_lattice(cfg["ids"], cfg["frozen"], cfg["cell_type"]); o.set_lattice(cfg["ids"], cfg["frozen"], cfg["cell_type"])
        g.step(2); o.step(2)
        np.testing.assert_array_equal(g.get_lattice(), o.get_lattice())
        sg, so = g.get_cell_stats(), o.get_cell_stats()
        for k in so:
            np.testing.assert_array_equal(sg[k], so[k])


@pytest.mark.parametrize("name,dims", [("C4", (256, 256, 256)), ("C5", (4096, 4096))])
def test_pinned_buffers_at_the_natural_threshold(pk, oracle_mod, name, dims):
    """2^24 sites: the slab path as a user meets it, with PINNED host buffers, whose copies really are asynchronous (a
    pageable source holds the host up, which would hide an ordering mistake between the transfer stream and the kernels).
    State after cpm_set_lattice, the read-back into a pinned buffer, and one MCS equal the oracle's, over four calls
    that alternate between two lattices."""
    import torch
    import cpm_inputs as ci
    cfg = ci.make_config(name, dims=dims)
    p = dict(cfg["params"]); p["subsection"] = 0
    g = pk.CPM(cfg["dims"], max_cells=cfg["max_cells"], **p)
    o = oracle_mod.Oracle(cfg["dims"], max_cells=cfg["max_cells"], **p)
    # two different lattices taken in turns: the staging buffers still hold the other one from the call before, so a kernel
    # that ran ahead of its slab's copy would pack stale words
    ids_b = np.ascontiguousarray(np.roll(cfg["ids"], (7, 5), axis=(0, -1)))
    fz_b = np.ascontiguousarray(np.roll(cfg["frozen"], (7, 5), axis=(0, -1))) if cfg["frozen"] is not None else None
    inputs, want = [], []
    for ids, fz in ((cfg["ids"], cfg["frozen"]), (ids_b, fz_b)):
        o.set_lattice(ids, fz, cfg["cell_type"])
        want.append(o.get_cell_stats())
        inputs.append((torch.from_numpy(ids.view(np.int32).reshape(-1)).pin_memory(),
                       torch.from_numpy(fz.reshape(-1)).pin_memory() if fz is not None else None))
    ct_h = torch.from_numpy(cfg["cell_type"]).pin_memory()
    out_h = torch.empty(inputs[0][0].numel(), dtype=torch.int32).pin_memory()
    for rep in (0, 1, 0, 1):
        ids_h, fz_h = inputs[rep]
        out_h.fill_(-1)
        g.set_lattice(ids_h, fz_h, ct_h)
        sg = g.get_cell_stats()
        for k in want[rep]:
            np.testing.assert_array_equal(sg[k], want[rep][k], err_msg="%s, lattice %d" % (k, rep))
        g.get_lattice(out_h)
        assert torch.equal(out_h, ids_h)
    g.set_mcs(0); g.step(1); o.step(1)     # both hold the second lattice
    g.get_lattice(out_h)
    np.testing.assert_array_equal(out_h.numpy().view(np.uint32).reshape(cfg["ids"].shape), o.get_lattice())
