"""GPU parity: libpic (CUDA, through the C ABI) against the CPU oracle, element by element, on the
seeded inputs of the five BASELINE.json configs at sizes the oracle finishes in seconds that
still span many tiles and ragged tails, plus the arranger's edge and degenerate cases.
Full-size runs live in test_gpu_fullsize.py."""
import numpy as np
import pytest

import oracle
import paper_2603_24508_b200 as pic
from paper_2603_24508_b200 import workloads
from parity_util import compare, make_pair, run_bulk, run_stepwise

pytestmark = pytest.mark.gpu

VARIANTS = [
    pytest.param({"fused": 0}, id="split"),
    pytest.param({"fused": 0, "tile_scatter": 0}, id="split-destscatter"),
    pytest.param({"fused": 1}, id="fused"),
    pytest.param({"fused": 1, "fused_stages": 2}, id="fused-2stage"),
    pytest.param({"fused": 1, "fused_tma": 0}, id="fused-plainloads"),
]


@pytest.mark.parametrize("options", VARIANTS)
def test_config1_full_200_steps(options):
    """configs[0]: 1,024 periodic cells x 64 = 65,536 electrons, 200 steps, arrange every step."""
    inp = workloads.make(1)
    run_stepwise(inp, 200, options=options)


@pytest.mark.parametrize("options", VARIANTS)
def test_config1_bulk_equals_stepwise(options):
    inp = workloads.make(1)
    run_bulk(inp, 200, options=options)


@pytest.mark.parametrize("options", VARIANTS)
def test_config2_reduced_absorbing(options):
    """configs[1] shape (absorbing walls, 160 ppc, 85 deg) on 2,048 cells: 327,680 particles, ragged tail."""
    inp = workloads.make(2, nc=2048)
    sim, states = run_stepwise(inp, 100, options=options, check_every=5)
    assert states[0].wall.sum() > 0  # the walls did absorb something, so compaction was exercised


@pytest.mark.parametrize("options", VARIANTS)
def test_config3_reduced_two_species(options):
    """configs[2] shape: electrons + D+ (q/m = 1/3672), sheath field, absorbing walls, 200 ppc."""
    inp = workloads.make(3, nc=1000)
    run_stepwise(inp, 60, options=options, check_every=4)


@pytest.mark.parametrize("options", VARIANTS + [pytest.param({"fused": 1, "species_streams": 0}, id="fused-one-stream")])
@pytest.mark.parametrize("chunk", [1, 7])
def test_push_all_species_on_their_own_streams(options, chunk):
    """pic_push_all: electrons, D+ and a neutral species stepped together (each species on an internal stream of its
    own, kernels overlapping) -- every species must match its oracle bit for bit, the call must leave everything ordered
    on the sim's stream (the comparison reads the buffers through that stream), and calls may be interleaved with
    per-species pic_push / pic_arrange."""
    inp = workloads.make(3, nc=1500)
    e = inp["species"][0]
    inp["species"].append(dict(e, qm=0.0, x=e["x"].copy(), vx=e["vx"].copy(), vy=e["vy"].copy(), vz=e["vz"].copy(),
                               cell=e["cell"].copy()))
    sim, states = make_pair(inp, options=options)
    done = 0
    while done < 42:
        pic.pic_push_all(sim, chunk)
        for st in states:
            st.push(chunk)
        done += chunk
        if done == 14:  # one species alone in between, then an explicit arrange of another
            pic.pic_push(sim.species[1], 2)
            states[1].push(2)
            pic.pic_arrange(sim.species[2])
            states[2].arrange()
        if done % 14 == 0:
            for si, (sp, st) in enumerate(zip(sim.species, states)):
                compare(sp, st, where=f"push_all step {done} species {si}", counts=True, nc=inp["nc"])
    pic.pic_sync(sim)
    assert states[0].wall.sum() > 0


def test_push_all_single_species_and_errors():
    inp = workloads.make(1, nc=256, ppc=32)
    sim, states = make_pair(inp)
    pic.pic_push_all(sim, 5)
    states[0].push(5)
    compare(sim.species[0], states[0], where="push_all, one species", counts=True, nc=inp["nc"])
    with pytest.raises(pic.PicError):
        pic.pic_push_all(sim, -1)


@pytest.mark.parametrize("options", VARIANTS)
def test_config4_reduced_periodic(options):
    """configs[3] shape: periodic, 100 ppc, 16 modes; 4,099 cells (odd, prime) -> 409,900 particles."""
    inp = workloads.make(4, nc=4099)
    run_stepwise(inp, 50, options=options, check_every=5)


@pytest.mark.parametrize("options", VARIANTS)
def test_config5_reduced_sort_stress(options):
    """configs[4] shape: 100x density contrast, v_th = 4, arrange every 10 steps, dead particles stay
    flagged in place between arranges (compared slot by slot)."""
    inp = workloads.make(5, nc=4096)
    sim, states = run_stepwise(inp, 40, options=options, check_every=1)
    w, used_general = pic.pic_arrange_info(sim.species[0])
    assert used_general == 0


def test_explicit_arrange_and_no_auto_arrange():
    """arrange_every = 0: pushes never arrange; pic_arrange() on demand; arranging twice is the identity."""
    inp = workloads.make(2, nc=512)
    sim, (st,) = make_pair(inp, arrange_every=0)
    sp = sim.species[0]
    for k in range(7):
        pic.pic_push(sp, 3)
        st.push(3)
        compare(sp, st, where=f"push block {k}")
        pic.pic_arrange(sp)
        st.arrange()
        compare(sp, st, where=f"arrange {k}", counts=True, nc=inp["nc"])
    pic.pic_arrange(sp)
    st.arrange()
    compare(sp, st, where="second arrange", counts=True, nc=inp["nc"])
    with pytest.raises(pic.PicError):
        pic.pic_push(sp, 1)
        pic.pic_cell_counts(sp, inp["nc"])  # stale after a push -> PIC_ESTATE


def test_general_path_unsorted_input():
    """An initial state that is NOT grouped by cell takes the general (radix) path on the first arrange."""
    inp = workloads.make(1, nc=300, ppc=37)
    rng = np.random.default_rng(7)
    s = inp["species"][0]
    perm = rng.permutation(len(s["x"]))
    for k in ("x", "vx", "vy", "vz", "cell"):
        s[k] = np.ascontiguousarray(s[k][perm])
    sim, (st,) = make_pair(inp)
    sp = sim.species[0]
    pic.pic_push(sp, 1)
    st.push(1)
    compare(sp, st, where="first arrange (general)", counts=True, nc=inp["nc"])
    assert pic.pic_arrange_info(sp)[1] == 1
    pic.pic_push(sp, 5)
    st.push(5)
    compare(sp, st, where="later arranges (fast)", counts=True, nc=inp["nc"])
    assert pic.pic_arrange_info(sp)[1] == 0


def test_general_path_large_displacement():
    """Many pushes without arranging: the displacement bound exceeds the fast path's limit."""
    inp = workloads.make(5, nc=2048)
    sim, (st,) = make_pair(inp, arrange_every=0)
    sp = sim.species[0]
    pic.pic_push(sp, 150)
    st.push(150)
    pic.pic_arrange(sp)
    st.arrange()
    compare(sp, st, where="arrange after 150 free steps", counts=True, nc=inp["nc"])
    assert pic.pic_arrange_info(sp)[1] == 1


def test_general_path_without_workspace_reports():
    inp = workloads.make(1, nc=64, ppc=8)
    s = inp["species"][0]
    perm = np.random.default_rng(3).permutation(len(s["x"]))
    for k in ("x", "vx", "vy", "vz", "cell"):
        s[k] = np.ascontiguousarray(s[k][perm])
    sim, _ = make_pair(inp, workspace=None)
    pic.pic_push(sim.species[0], 1)
    with pytest.raises(pic.PicError) as e:
        pic.pic_wall_flux(sim.species[0])
    assert e.value.status == pic.PIC_ECAPACITY


@pytest.mark.parametrize("n", [0, 1, 2, 3, 31, 32, 33, 511, 513])
@pytest.mark.parametrize("boundary", [workloads.PERIODIC, workloads.ABSORBING])
def test_tiny_and_ragged(n, boundary):
    rng = np.random.default_rng(100 + n)
    nc = 5
    cell = np.sort(rng.integers(0, nc, n)).astype(np.int32)
    x = cell + rng.random(n)
    x = np.where(np.floor(x) != cell, np.nextafter(cell + 1.0, 0), x)
    v = 6.0 * rng.standard_normal((3, n))
    inp = dict(nc=nc, dx=1.0, dt=0.1, boundary=boundary, E=rng.uniform(-1, 1, nc + 1), B=np.array([0.3, -1.0, 2.0]),
               arrange_every=1, species=[dict(qm=-1.0, x=x, vx=v[0], vy=v[1], vz=v[2], cell=cell)])
    for options in ({"fused": 0}, {"fused": 1}):
        run_stepwise(inp, 12, options=options)


def test_single_cell_and_all_absorbed():
    rng = np.random.default_rng(5)
    n = 1000
    cell = np.zeros(n, dtype=np.int32)
    x = rng.random(n)
    inp = dict(nc=1, dx=1.0, dt=0.1, boundary=workloads.ABSORBING, E=np.array([0.1, -0.2]), B=np.array([0.0, 2.0, 0.0]),
               arrange_every=1,
               species=[dict(qm=-1.0, x=x, vx=3.0 * rng.standard_normal(n), vy=rng.standard_normal(n),
                             vz=rng.standard_normal(n), cell=cell)])
    sim, (st,) = run_stepwise(inp, 40)
    assert st.n + int(st.wall.sum()) == n
    # periodic single cell: every particle wraps within the same cell
    inp["boundary"] = workloads.PERIODIC
    inp["E"] = np.array([0.1, 0.1])
    run_stepwise(inp, 20)


def test_dx_not_one_and_three_component_B():
    """dx != 1 exercises the inv_dx products and the clamp reading S8; B with a z component."""
    rng = np.random.default_rng(11)
    nc, ppc, dx = 257, 21, 0.37
    cell = np.repeat(np.arange(nc, dtype=np.int32), ppc)
    x = (cell + rng.random(nc * ppc)) * dx
    inv = 1.0 / dx
    ok = np.minimum(np.floor(x * inv), nc - 1) == cell
    x = x[ok]; cell = cell[ok]
    keep = x < nc * dx
    x = x[keep]; cell = cell[keep]
    n = len(x)
    v = rng.standard_normal((3, n))
    for boundary in (workloads.PERIODIC, workloads.ABSORBING):
        E = rng.uniform(-0.5, 0.5, nc + 1)
        if boundary == workloads.PERIODIC:
            E[nc] = E[0]
        inp = dict(nc=nc, dx=dx, dt=0.05, boundary=boundary, E=E, B=np.array([1.5, 1.25, 0.5]), arrange_every=1,
                   species=[dict(qm=-1.0, x=x, vx=v[0], vy=v[1], vz=v[2], cell=cell)])
        for options in ({"fused": 0}, {"fused": 1}):
            run_stepwise(inp, 30, options=options)


def test_create_rejects_bad_state():
    inp = workloads.make(1, nc=16, ppc=4)
    s = inp["species"][0]
    s["cell"] = s["cell"].copy()
    s["cell"][5] += 1  # cell != floor(x)
    with pytest.raises(pic.PicError) as e:
        make_pair(inp)
    assert e.value.status == pic.PIC_ESTATE


def test_wall_flux_recent_and_step_counters():
    inp = workloads.make(2, nc=256)
    sim, (st,) = make_pair(inp)
    sp = sim.species[0]
    pic.pic_push(sp, 10)
    a = pic.pic_wall_flux(sp)
    pic.pic_push(sp, 15)
    b = pic.pic_wall_flux(sp)
    st.push(25)
    assert b["left_total"] == int(st.wall[0]) and b["right_total"] == int(st.wall[1])
    assert a["left_recent"] == a["left_total"] and b["left_recent"] == b["left_total"] - a["left_total"]
    assert b["right_recent"] == b["right_total"] - a["right_total"]
    assert (a["steps_recent"], b["steps_recent"], b["steps_total"]) == (10, 15, 25)
    assert pic.pic_step_count(sp) == 25


def test_run_host_end_to_end():
    """pic_run_host: the C-ABI call with HOST buffers (the one bench.py's e2e leg times)."""
    import ctypes as C
    inp = workloads.make(2, nc=512)
    s = inp["species"][0]
    st = oracle.State(s["x"], s["vx"], s["vy"], s["vz"], s["cell"], nc=inp["nc"], dx=inp["dx"], dt=inp["dt"],
                      boundary=inp["boundary"], E=inp["E"], qm=s["qm"], B=inp["B"], arrange_every=1)
    st.push(20)
    arrs = [np.array(s[k]) for k in ("x", "vx", "vy", "vz", "cell")]
    n_out, wl, wr = pic.pic_run_host(nc=inp["nc"], dx=inp["dx"], dt=inp["dt"], boundary=inp["boundary"], E_nodes=inp["E"],
                                     B=inp["B"], species=[dict(qm=s["qm"], arrays=arrs, arrange_every=1)], nsteps=20)[0]
    assert n_out == st.n and (wl, wr) == (int(st.wall[0]), int(st.wall[1]))
    for a, o in zip(arrs, st.live()):
        assert np.array_equal(a[:n_out], o)


def test_memory_pool_is_reused_and_trimmed():
    """The library's device memory comes from a pool that keeps freed blocks ("allocate once, keep
    resident"): repeated pic_run_host calls give the same result from the cached arena, the process holds the memory
    in between, and pic_trim_memory returns it to the driver."""
    import torch
    inp = workloads.make(4, nc=20000)  # 2 M particles: an arena of ~150 MB
    s = inp["species"][0]
    st = oracle.State(s["x"], s["vx"], s["vy"], s["vz"], s["cell"], nc=inp["nc"], dx=inp["dx"], dt=inp["dt"],
                      boundary=inp["boundary"], E=inp["E"], qm=s["qm"], B=inp["B"], arrange_every=1)
    st.push(5)
    pic.pic_trim_memory()
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        arrs = [np.array(s[k]) for k in ("x", "vx", "vy", "vz", "cell")]
        n_out, _, _ = pic.pic_run_host(nc=inp["nc"], dx=inp["dx"], dt=inp["dt"], boundary=inp["boundary"], E_nodes=inp["E"],
                                       B=inp["B"], species=[dict(qm=s["qm"], arrays=arrs, arrange_every=1)], nsteps=5)[0]
        assert n_out == st.n
        for a, o in zip(arrs, st.live()):
            assert np.array_equal(a[:n_out], o)
    held = free0 - torch.cuda.mem_get_info()[0]
    assert held >= 100 << 20, f"the pool should still hold the arena, holds {held} bytes"
    pic.pic_trim_memory()
    assert free0 - torch.cuda.mem_get_info()[0] < 32 << 20, "pic_trim_memory did not return the cached memory"


@pytest.mark.parametrize("config,kw,steps,pinned", [(3, dict(nc=1500), 25, True), (5, dict(nc=2048), 23, False)])
def test_run_host_two_species_and_pinned_buffers(config, kw, steps, pinned):
    """pic_run_host with several species in one call (one device arena, D2H on a second stream), pinned torch
    buffers or plain numpy arrays; config 5 ends between two arranges, so flagged-dead particles come back in place;
    and the binding refuses arrays it cannot hand to the C side."""
    import torch
    inp = workloads.make(config, **kw)
    ae = inp["arrange_every"]
    species, states = [], []
    for s in inp["species"]:
        st = oracle.State(s["x"], s["vx"], s["vy"], s["vz"], s["cell"], nc=inp["nc"], dx=inp["dx"], dt=inp["dt"],
                          boundary=inp["boundary"], E=inp["E"], qm=s["qm"], B=inp["B"], arrange_every=ae)
        st.push(steps)
        states.append(st)
        arrs = [np.array(s[k]) for k in ("x", "vx", "vy", "vz", "cell")]
        if pinned:
            arrs = [torch.from_numpy(a).pin_memory() for a in arrs]
        species.append(dict(qm=s["qm"], arrays=arrs, arrange_every=ae))
    if config == 5:  # a second species of the same shape, so that both kinds of state come back from one call
        species.append(dict(qm=species[0]["qm"], arrays=[np.array(inp["species"][0][k]) for k in ("x", "vx", "vy", "vz", "cell")],
                            arrange_every=ae))
        states.append(states[0])
    res = pic.pic_run_host(nc=inp["nc"], dx=inp["dx"], dt=inp["dt"], boundary=inp["boundary"], E_nodes=inp["E"], B=inp["B"],
                           species=species, nsteps=steps)
    for (n_out, wl, wr), sp, st in zip(res, species, states):
        assert n_out == st.n and (wl, wr) == (int(st.wall[0]), int(st.wall[1]))
        for a, o in zip(sp["arrays"], st.live()):
            a = a.numpy() if hasattr(a, "numpy") else a
            assert np.array_equal(a[:n_out], o)
    bad = [np.array(inp["species"][0][k]) for k in ("x", "vx", "vy", "vz", "cell")]
    bad[1] = bad[1].astype(np.float32)
    with pytest.raises(ValueError):
        pic.pic_run_host(nc=inp["nc"], dx=inp["dx"], dt=inp["dt"], boundary=inp["boundary"], E_nodes=inp["E"], B=inp["B"],
                         species=[dict(qm=-1.0, arrays=bad, arrange_every=ae)], nsteps=1)
    bad[1] = bad[1].astype(np.float64)[:-1]
    with pytest.raises(ValueError):
        pic.pic_run_host(nc=inp["nc"], dx=inp["dx"], dt=inp["dt"], boundary=inp["boundary"], E_nodes=inp["E"], B=inp["B"],
                         species=[dict(qm=-1.0, arrays=bad, arrange_every=ae)], nsteps=1)


@pytest.mark.parametrize("config,kw,steps", [(1, {}, 40), (2, dict(nc=2048), 40), (3, dict(nc=1000), 30),
                                             (4, dict(nc=4099), 30)])
def test_fused_step_is_the_one_that_runs(config, kw, steps):
    """Configs 1-4 (arrange every step, |dcell| <= 1): every step is taken by the fused kernels,
    none is redone by the guarded split chain."""
    inp = workloads.make(config, **kw)
    sim, states = run_stepwise(inp, steps, options={"fused": 1}, check_every=10)
    for sp in sim.species:
        info = pic.pic_fused_info(sp)
        assert info["active"] == 1 and info["decline_reasons"] == 0, info
        assert pic.pic_arrange_info(sp)[1] == 0


@pytest.mark.parametrize("knobs", [
    {"fused_cells_per_cta": 1}, {"fused_cells_per_cta": 3, "fused_rows": 12}, {"fused_cells_per_cta": 256},
    {"fused_rows": 16}, {"fused_cells_per_cta": 33, "fused_rows": 8}, {"fused_cells_per_cta": 7},
    {"fused_cells_per_cta": 16, "fused_taper": 3}, {"fused_cells_per_cta": 64, "fused_taper": 1},
    {"fused_cells_per_cta": 5, "fused_taper": 2}, {"fused_cells_per_cta": 256, "fused_taper": 3},
])
@pytest.mark.parametrize("config,kw", [(4, dict(nc=4099)), (2, dict(nc=1500))])
def test_fused_knobs_do_not_change_results(knobs, config, kw):
    """Cells per CTA, the tapered chunk schedule and rows per tile only move the tile / chunk borders (halo cells,
    deferred right-movers, carried counts land elsewhere); results stay bit-identical."""
    inp = workloads.make(config, **kw)
    sim, _ = run_stepwise(inp, 12, options={"fused": 1, **knobs}, check_every=3)
    info = pic.pic_fused_info(sim.species[0])
    assert info["decline_reasons"] == 0, info


def test_fused_declines_when_a_cell_does_not_fit_and_split_redoes_the_step():
    """Tiles of 8 rows (256 slots) against 300 particles per cell: the fused step aborts on the
    device, the guarded split kernels redo it from the untouched source buffers."""
    inp = workloads.make(2, nc=512, ppc=300)
    sim, _ = run_stepwise(inp, 6, options={"fused": 1, "fused_rows": 8}, check_every=1)
    info = pic.pic_fused_info(sim.species[0])
    assert info["decline_reasons"] & 2, info


def test_fused_large_cells_take_the_wide_tiles():
    """300 particles per cell: 16-row tiles chosen automatically."""
    inp = workloads.make(2, nc=512, ppc=300)
    sim, _ = run_stepwise(inp, 6, options={"fused": 1}, check_every=1)
    info = pic.pic_fused_info(sim.species[0])
    assert info["decline_reasons"] == 0 and info["active"] == 1 and info["stage_slots"] == 512, info


def test_fused_declines_on_a_two_cell_jump():
    """One particle fast enough to cross two cells in a step: the fused step declines (reason 1),
    the split path takes over for good, results unchanged."""
    inp = workloads.make(1, nc=512, ppc=40)
    s = inp["species"][0]
    s["vx"] = s["vx"].copy()
    s["vx"][12345] = 23.0
    sim, _ = run_stepwise(inp, 8, options={"fused": 1}, check_every=1)
    info = pic.pic_fused_info(sim.species[0])
    assert info["decline_reasons"] & 1 and info["active"] == 0, info


def test_fused_empty_cells_and_sparse_density():
    """Many empty cells and cells of very different size (config-5 density, slow particles so the
    fused step applies): empty tiles, empty halo cells, tiles of many cells."""
    inp = workloads.make(5, nc=2048, n_total=150000)
    for s in inp["species"]:
        for k in ("vx", "vy", "vz"):
            s[k] = s[k] * 0.25
    inp["arrange_every"] = 1
    sim, states = run_stepwise(inp, 25, options={"fused": 1}, check_every=1)
    assert (states[0].count == 0).any()
    info = pic.pic_fused_info(sim.species[0])
    assert info["decline_reasons"] == 0, info


def test_fused_declined_mid_run_is_redone_at_the_next_sync():
    """Fused steps are enqueued without a fallback behind them; a step that declines freezes the state and is
    redone (with all later steps) by the split kernels at the next synchronising call.  Here one particle turns
    fast enough to jump two cells only after a few gyration steps, in the middle of one pic_push(sp, 20)."""
    inp = workloads.make(1, nc=512, ppc=40)
    s = inp["species"][0]
    for k in ("vx", "vy", "vz"):
        s[k] = s[k].copy()
    p = 7777
    s["vx"][p], s["vy"][p], s["vz"][p] = 0.0, 0.0, 26.0
    # oracle: first step at which that particle moves two cells or more
    probe = oracle.State(s["x"][p:p + 1], s["vx"][p:p + 1], s["vy"][p:p + 1], s["vz"][p:p + 1], s["cell"][p:p + 1], nc=inp["nc"],
                         dx=inp["dx"], dt=inp["dt"], boundary=inp["boundary"], E=inp["E"], qm=s["qm"], B=inp["B"], arrange_every=0)
    first = None
    for k in range(1, 21):
        c0 = int(probe.cell[0])
        probe.push(1)
        d = abs(int(probe.cell[0]) - c0)
        if min(d, inp["nc"] - d) >= 2:
            first = k
            break
    assert first is not None and 2 <= first <= 15, first
    sim, (st,) = make_pair(inp, options={"fused": 1})
    sp = sim.species[0]
    pic.pic_push(sp, 20)
    st.push(20)
    compare(sp, st, where="bulk 20 with a declined fused step inside", counts=True, nc=inp["nc"])
    info = pic.pic_fused_info(sp)
    assert info["decline_reasons"] & 1 and info["active"] == 0, info
    assert pic.pic_step_count(sp) == 20
    pic.pic_push(sp, 5)
    st.push(5)
    compare(sp, st, where="after the switch to the split path", counts=True, nc=inp["nc"])


@pytest.mark.parametrize("boundary", [workloads.PERIODIC, workloads.ABSORBING])
def test_tile_scatter_declines_on_sparse_tiles(boundary):
    """About one particle per cell: a tile of 2,048 slots spans more cells than a window holds, the
    tile-ranked scatter declines and the destination-driven scatter takes the arrange (same result)."""
    rng = np.random.default_rng(21)
    nc = 6000
    cell = np.sort(rng.integers(0, nc, 7000)).astype(np.int32)
    x = cell + rng.random(len(cell))
    x = np.where(np.floor(x) != cell, np.nextafter(cell + 1.0, 0), x)
    v = 3.0 * rng.standard_normal((3, len(cell)))
    E = rng.uniform(-0.2, 0.2, nc + 1)
    if boundary == workloads.PERIODIC:
        E[nc] = E[0]
    inp = dict(nc=nc, dx=1.0, dt=0.1, boundary=boundary, E=E, B=np.array([1.0, 1.0, 0.0]), arrange_every=3,
               species=[dict(qm=-1.0, x=x, vx=v[0], vy=v[1], vz=v[2], cell=cell)])
    run_stepwise(inp, 12, options={"fused": 0})


def test_tile_scatter_wraps_and_large_displacements():
    """Periodic grid, arrange every 7 steps with fast particles: windows that straddle the ends of the grid."""
    inp = workloads.make(5, nc=1024, n_total=200000)
    inp["boundary"] = workloads.PERIODIC
    inp["E"][inp["nc"]] = inp["E"][0]
    inp["arrange_every"] = 7
    sim, _ = run_stepwise(inp, 28, options={"fused": 0})
    assert pic.pic_arrange_info(sim.species[0])[1] == 0


DEP_RTOL = 1e-12  # north_star tolerance; the GPU sums each cell with a fixed tree, the oracle sequentially


def _check_deposit(sp, st, weight, where):
    rho = pic.pic_deposit(sp, weight).cpu().numpy()
    ref = st.deposit(weight)
    scale = np.maximum(np.abs(ref), abs(weight))
    assert np.all(np.abs(rho - ref) <= DEP_RTOL * scale), f"{where}: deposition differs, max {np.max(np.abs(rho - ref) / scale)}"
    return rho


@pytest.mark.parametrize("config,kw,fused", [(1, {}, 1), (2, dict(nc=2048), 1), (4, dict(nc=4099), 0), (5, dict(nc=4096), 1)])
def test_deposit_matches_oracle(config, kw, fused):
    """pic_deposit on the arranged state after every arranging step: all nodes within 1e-12 relative
    (to max(|rho_j|, |weight|)); total charge = weight * n_live."""
    inp = workloads.make(config, **kw)
    sim, states = make_pair(inp, options={"fused": fused})
    ae = inp["arrange_every"]
    for step in range(1, 21):
        for sp, st in zip(sim.species, states):
            pic.pic_push(sp, 1)
            st.push(1)
        if step % ae == 0:
            for sp, st in zip(sim.species, states):
                rho = _check_deposit(sp, st, -0.75, f"config {config} step {step}")
                tot = rho[:-1].sum() if inp["boundary"] == workloads.PERIODIC else rho.sum()
                assert abs(tot - (-0.75) * st.n) <= 1e-10 * 0.75 * st.n
    pic.pic_sync(sim)


def test_deposit_two_species_accumulate_and_state_errors():
    inp = workloads.make(3, nc=1000)
    sim, states = make_pair(inp)
    for sp, st in zip(sim.species, states):
        pic.pic_push(sp, 3)
        st.push(3)
    rho = pic.pic_deposit(sim.species[0], -1.0)
    rho = pic.pic_deposit(sim.species[1], +1.0, rho=rho, accumulate=True).cpu().numpy()
    ref = states[0].deposit(-1.0) + states[1].deposit(+1.0)
    scale = np.maximum(np.abs(states[0].deposit(-1.0)), 1.0)
    assert np.all(np.abs(rho - ref) <= 1e-12 * scale)
    # not arranged -> PIC_ESTATE
    inp5 = workloads.make(5, nc=512)
    sim5, _ = make_pair(inp5)
    pic.pic_push(sim5.species[0], 1)
    with pytest.raises(pic.PicError) as e:
        pic.pic_deposit(sim5.species[0], 1.0)
    assert e.value.status == pic.PIC_ESTATE


def test_deposit_empty_cells_tiny_and_dx():
    rng = np.random.default_rng(13)
    nc, dx = 40, 0.37
    cell = np.sort(rng.choice(nc, size=25, replace=True)).astype(np.int32)
    x = (cell + rng.random(len(cell))) * dx
    ok = np.minimum(np.floor(x * (1.0 / dx)), nc - 1) == cell
    x, cell = x[ok], cell[ok]
    v = rng.standard_normal((3, len(x)))
    for boundary in (workloads.PERIODIC, workloads.ABSORBING):
        E = np.zeros(nc + 1)
        inp = dict(nc=nc, dx=dx, dt=0.05, boundary=boundary, E=E, B=np.array([0.0, 1.0, 0.0]), arrange_every=1,
                   species=[dict(qm=-1.0, x=x, vx=v[0], vy=v[1], vz=v[2], cell=cell)])
        sim, (st,) = make_pair(inp)
        _check_deposit(sim.species[0], st, 2.5, "initial state")
        pic.pic_push(sim.species[0], 4)
        st.push(4)
        _check_deposit(sim.species[0], st, 2.5, "after 4 steps")


def test_neutral_species_qm_zero():
    """Neutral species (`nmove` / `narrj`) are the same kernels with q/m = 0: ballistic motion,
    same arranger; three species side by side as in the paper's ionisation case (e-, D+, D)."""
    inp = workloads.make(3, nc=600)
    neutral = dict(inp["species"][1])
    neutral["qm"] = 0.0
    neutral["name"] = "D"
    inp["species"].append(neutral)
    sim, states = run_stepwise(inp, 20, check_every=5)
    v0 = neutral["vx"]
    assert np.array_equal(np.sort(states[2].vx[:states[2].n]), np.sort(v0)[:states[2].n]) or states[2].n < len(v0)
    for sp in sim.species:
        assert pic.pic_fused_info(sp)["decline_reasons"] == 0


@pytest.mark.parametrize("seed", range(6))
def test_random_api_sequences(seed):
    """Random interleavings of pic_push(k), pic_arrange, pic_set_field, pic_wall_flux, pic_deposit and full state
    comparisons, for every arrange_every rule, both boundaries, with and without a particle that makes the fused
    step decline somewhere in the middle: the host bookkeeping (buffer parity, step counter, deferred check of
    fused steps, wall counter intervals) must stay in lock-step with the oracle."""
    rng = np.random.default_rng(1000 + seed)
    boundary = workloads.PERIODIC if seed % 2 == 0 else workloads.ABSORBING
    ae = (1, 1, 3, 0, 1, 2)[seed]
    nc, ppc = 257, 24
    cell = np.repeat(np.arange(nc, dtype=np.int32), ppc)
    x = cell + rng.random(len(cell))
    x = np.where(np.floor(x) != cell, np.nextafter(cell + 1.0, 0), x)
    v = rng.standard_normal((3, len(cell)))
    if seed in (1, 4):
        v[2, 1234] = 24.0  # turns into vx > 10 after a few gyrations: a two-cell jump, the fused step declines
    def field():
        E = rng.uniform(-0.3, 0.3, nc + 1)
        if boundary == workloads.PERIODIC:
            E[nc] = E[0]
        return E
    inp = dict(nc=nc, dx=1.0, dt=0.1, boundary=boundary, E=field(), B=np.array([1.4, 1.4, 0.3]), arrange_every=ae,
               species=[dict(qm=-1.0, x=x, vx=v[0], vy=v[1], vz=v[2], cell=cell)])
    sim, (st,) = make_pair(inp)
    sp = sim.species[0]
    arranged = False  # the oracle fills count / offset at its first arrange only
    last_flux_steps = 0
    for op_i in range(40):
        op = rng.choice(["push", "push", "push", "arrange", "field", "flux", "deposit", "compare"])
        if op == "push":
            k = int(rng.integers(1, 5))
            pic.pic_push(sp, k)
            st.push(k)
            arranged = ae > 0 and st.steps % ae == 0
        elif op == "arrange":
            pic.pic_arrange(sp)
            st.arrange()
            arranged = True
        elif op == "field":
            E = field()
            pic.pic_set_field(sim, E)
            st.E = np.ascontiguousarray(E)
        elif op == "flux":
            wf = pic.pic_wall_flux(sp)
            assert (wf["left_total"], wf["right_total"]) == (int(st.wall[0]), int(st.wall[1]))
            assert wf["steps_recent"] == st.steps - last_flux_steps and wf["steps_total"] == st.steps
            last_flux_steps = st.steps
        elif op == "deposit" and arranged:
            _check_deposit(sp, st, 1.5, f"seed {seed} op {op_i}")
        elif op == "compare":
            wf = compare(sp, st, where=f"seed {seed} op {op_i}", counts=arranged, nc=nc)
            last_flux_steps = st.steps
    compare(sp, st, where=f"seed {seed} end", counts=arranged, nc=nc)
    pic.pic_sync(sim)
    if seed in (1, 4) and st.steps >= 12:
        assert pic.pic_fused_info(sp)["decline_reasons"] & 1, "the fast particle should have made a fused step decline"


def test_fused_path_comes_back_after_the_cause_is_gone():
    """One particle far too fast for the fused step (2.5 cells per step) on an absorbing grid: the fused step
    declines, the split kernels carry the run, the particle is absorbed at the wall, and 16 steps later a
    synchronising call switches the fused path back on.  Parity throughout."""
    inp = workloads.make(2, nc=256, ppc=40)
    s = inp["species"][0]
    for k in ("vx", "vy", "vz"):
        s[k] = s[k].copy()
    p = 40 * 200 + 3  # a particle in cell 200 heading for the right wall
    s["vx"][p], s["vy"][p], s["vz"][p] = 25.0, 0.0, 0.0
    inp["B"] = np.array([2.0, 0.0, 0.0])  # B along x: vx is not rotated away
    sim, (st,) = make_pair(inp, options={"fused": 1})
    sp = sim.species[0]
    seen_off = seen_back = False
    for step in range(1, 71):
        pic.pic_push(sp, 1)
        st.push(1)
        if step % 5 == 0:
            compare(sp, st, where=f"step {step}", counts=True, nc=inp["nc"])
            info = pic.pic_fused_info(sp)
            if info["active"] == 0:
                seen_off = True
            elif seen_off:
                seen_back = True
    assert seen_off and seen_back, "fused path should have declined and then come back"
    assert pic.pic_fused_info(sp)["decline_reasons"] & 1


def test_bench_guard_fires_when_a_fused_step_declines_in_the_timed_region():
    """bench.py must not be able to time skipped work: a particle that jumps two cells a few steps into the timed
    region makes a fused step decline; the redo by the split kernels has to fall inside the timed region
    (pic_sync before the closing event), the line must say so ("invalid", fused_path) and the exit code is 3."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    inp = workloads.make(1)
    s = inp["species"][0]
    p, vz = 7777, 26.0
    probe = oracle.State(s["x"][p:p + 1], np.zeros(1), np.zeros(1), np.full(1, vz), s["cell"][p:p + 1], nc=inp["nc"],
                         dx=inp["dx"], dt=inp["dt"], boundary=inp["boundary"], E=inp["E"], qm=s["qm"], B=inp["B"], arrange_every=0)
    first = None
    for k in range(1, 24):
        c0 = int(probe.cell[0])
        probe.push(1)
        d = abs(int(probe.cell[0]) - c0)
        if min(d, inp["nc"] - d) >= 2:
            first = k
            break
    assert first is not None and 3 < first <= 23, f"the jump must fall inside the timed region (step {first})"
    cmd = [sys.executable, os.path.join(root, "bench.py"), "--config", "1", "--steps", "20", "--warmup", "3", "--no-e2e",
           "--no-cpu", "--no-deposit", "--debug-fast-particle", str(vz)]
    r = subprocess.run(cmd, capture_output=True, text=True, cwd=root, timeout=600)
    assert r.returncode == 3, (r.returncode, r.stderr[-2000:])
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["invalid"] is True and "declined" in line["invalid_reason"]
    fp = line["fused_path"]
    assert fp["expected"] and fp["split_mover_steps"] > 0 and fp["decline_reasons"][0] & 1 and fp["active_after"] == [0]
    # and the clean run carries the same keys with nothing declined
    r = subprocess.run(cmd[:-2], capture_output=True, text=True, cwd=root, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    fp = line["fused_path"]
    assert "invalid" not in line and fp["split_mover_steps"] == 0 and fp["fused_steps"] == 20 and fp["decline_reasons"] == [0]


@pytest.mark.parametrize("options", VARIANTS)
@pytest.mark.parametrize("config,kw,steps", [(2, dict(nc=1024), 30), (5, dict(nc=2048), 30), (4, dict(nc=1531), 20)])
def test_no_write_beyond_the_initial_slot_count(options, config, kw, steps):
    """compute-sanitizer is closed on this pool (profiles/r02_sanitizers.md), so the bound is checked by hand: the
    buffers are allocated with 333 spare slots filled with a sentinel; the particle count never grows, so no kernel
    of any path (fused, split, tile-ranked, destination-driven) may ever write a slot >= n0 of either buffer set."""
    import torch
    inp = workloads.make(config, **kw)
    pad = 333
    sim, states = make_pair(inp, capacity_pad=pad, options=options)
    sent_f, sent_i = -1.2345678e300, -77777
    n0s = []
    for sp, s in zip(sim.species, inp["species"]):
        n0 = len(s["x"])
        n0s.append(n0)
        for b in range(2):
            for t in sp.bufs[b][:4]:
                t[n0:].fill_(sent_f)
            sp.bufs[b][4][n0:].fill_(sent_i)
    torch.cuda.synchronize()
    for sp, st in zip(sim.species, states):
        pic.pic_push(sp, steps)
        st.push(steps)
        pic.pic_arrange(sp)
        st.arrange()
        compare(sp, st, where=f"config {config} with spare capacity", counts=True, nc=inp["nc"])
    pic.pic_sync(sim)
    for sp, n0 in zip(sim.species, n0s):
        for b in range(2):
            for t in sp.bufs[b][:4]:
                assert bool((t[n0:] == sent_f).all()), "a kernel wrote beyond the initial slot count"
            assert bool((sp.bufs[b][4][n0:] == sent_i).all()), "a kernel wrote beyond the initial slot count (cell)"
    pic.pic_destroy(sim)


def test_fused_queue_of_deferred_right_movers_grows_with_the_flow():
    """A beam drifting at 3 cells per 10 steps on top of v_th = 1: about a third of every cell's particles move right
    each step, more than the 32 the smallest queue of deferred right-movers holds.  The first fused step declines
    (reason 4), the split kernels carry on, and once the host has seen the device's count the fused step comes back
    with a larger queue -- results bit-identical throughout."""
    inp = workloads.make(2, nc=1024)
    s = inp["species"][0]
    s["vx"] = s["vx"] + 3.0
    inp["B"] = np.array([2.0, 0.0, 0.0])  # B along x: the drift is not rotated away
    sim, (st,) = make_pair(inp, options={"fused": 1, "kernel_timing": 1})
    sp = sim.species[0]
    pic.pic_push(sp, 1)
    st.push(1)
    compare(sp, st, where="first step", counts=True, nc=inp["nc"])
    info = pic.pic_fused_info(sp)
    assert info["decline_reasons"] & 4 and info["active"] == 0, info
    for k in range(18):
        pic.pic_push(sp, 1)
        st.push(1)
    compare(sp, st, where="after the split steps", counts=True, nc=inp["nc"])
    info = pic.pic_fused_info(sp)
    assert info["active"] == 1, info
    pic.pic_kernel_time(sim, "fused")
    pic.pic_kernel_time(sim, "mover")
    pic.pic_push(sp, 25)
    st.push(25)
    compare(sp, st, where="fused again with a larger queue", counts=True, nc=inp["nc"])
    assert pic.pic_kernel_time(sim, "fused")[1] == 25 and pic.pic_kernel_time(sim, "mover")[1] == 0
    assert pic.pic_fused_info(sp)["active"] == 1
