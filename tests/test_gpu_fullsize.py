"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (own
stream, default options: fused single-pass step where arrange_every == 1, TMA-staged E).

Three kinds of check (task contract, parity at full size):
  * the WHOLE run (every step of the config) element by element -- all five arrays, per-cell counts, offsets,
    slot count, wall counters -- against the oracle's threaded twin (oracle/oracle_omp.c, pinned bit-identical
    to the single-thread oracle by tests/test_oracle_omp.py); config 2 also against the single-thread oracle
    itself;
  * element by element against the oracle for the first steps of every config (the oracle needs
    about a second per 30-40 M pushes, so a few steps of 100 M particles is still seconds);
  * after the config's whole step count: on SAMPLED particles the oracle computes one by one
    (the mover acts on each particle independently, so the oracle follows a sample from its
    initial state through all steps without arranging; the GPU's final state must contain that
    exact particle, bit for bit, inside the slot range of its final cell), plus properties that
    hold at any size (grouped by cell, cell == floor(x*inv_dx), counts/offsets consistent,
    n_live + absorbed == n_0) and EXACT wall counts from an oracle run over the only particles
    that can reach a wall (those within `margin` cells of it; checked to be enough).
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2603_24508_b200 as pic
from paper_2603_24508_b200 import workloads
from parity_util import compare, make_pair

pytestmark = pytest.mark.gpu


def _bench_like_pair(inp):
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        sim, states = make_pair(inp, stream=stream)
    return sim, states, stream


@pytest.mark.parametrize("config,steps,check_every", [(2, 4, 1), (3, 3, 1), (4, 3, 1), (5, 10, 5)])
def test_fullsize_first_steps_elementwise(config, steps, check_every):
    inp = workloads.make(config)
    sim, states, _ = _bench_like_pair(inp)
    ae = inp["arrange_every"]
    for step in range(1, steps + 1):
        for sp, st in zip(sim.species, states):
            st.push(1)
        pic.pic_push_all(sim, 1)  # the call bench.py times
        if step % check_every == 0 or step == steps:
            for si, (sp, st) in enumerate(zip(sim.species, states)):
                compare(sp, st, where=f"config {config} full size, step {step} species {si}",
                        counts=(step % ae == 0), nc=inp["nc"])
    pic.pic_sync(sim)
    for sp in sim.species:
        assert pic.pic_arrange_info(sp)[1] == 0, "full-size run fell to the general arranger"
    if steps % ae == 0:  # arranged state: charge deposition at full size against the oracle (1e-12)
        for sp, st in zip(sim.species, states):
            rho = pic.pic_deposit(sp, -1.0).cpu().numpy()
            ref = st.deposit(-1.0)
            assert np.all(np.abs(rho - ref) <= 1e-12 * np.maximum(np.abs(ref), 1.0)), f"config {config}: deposition differs"
    pic.pic_destroy(sim)


def _oracle_subset(inp, s, idx, steps):
    """Oracle trajectories (no arranging: the mover is per-particle) of the particles idx."""
    st = oracle.State(s["x"][idx], s["vx"][idx], s["vy"][idx], s["vz"][idx], s["cell"][idx], nc=inp["nc"],
                      dx=inp["dx"], dt=inp["dt"], boundary=inp["boundary"], E=inp["E"], qm=s["qm"], B=inp["B"],
                      arrange_every=0)
    st.push(steps)
    return st


@pytest.mark.parametrize("config,margin", [(2, 2000), (3, 2000), (4, 0), (5, 6000)])
def test_fullsize_all_steps_sampled_and_properties(config, margin):
    inp = workloads.make(config)
    nc, steps, ae = inp["nc"], inp["steps"], inp["arrange_every"]
    assert steps % ae == 0
    sim, _states, _ = _bench_like_pair(inp)
    del _states
    for sp in sim.species:
        pic.pic_push(sp, steps)  # one call, as bench.py's e2e leg; the timed leg calls it step by step
    pic.pic_sync(sim)
    rng = np.random.default_rng(99 + config)
    for si, (sp, s) in enumerate(zip(sim.species, inp["species"])):
        n0 = len(s["x"])
        wf = pic.pic_wall_flux(sp)
        n_live = pic.pic_n_slots(sp)
        x, vx, vy, vz, cell = sp.state()
        count, offset = pic.pic_cell_counts(sp, nc)
        assert pic.pic_arrange_info(sp)[1] == 0
        # ---- properties that hold at any size
        assert n_live + wf["left_total"] + wf["right_total"] == n0
        assert int(offset[nc]) == n_live and int(count.sum()) == n_live
        assert np.array_equal(np.concatenate([[0], np.cumsum(count, dtype=np.int64)]), offset.astype(np.int64))
        assert bool((cell[1:] >= cell[:-1]).all()), "not grouped by cell"
        inv_dx = 1.0 / inp["dx"]
        cf = torch.clamp(torch.floor(x * inv_dx).to(torch.int32), max=nc - 1)
        assert bool((cf == cell).all()), "cell != floor(x*inv_dx)"
        assert bool(((x >= 0) & (x < nc * inp["dx"])).all())
        bc = torch.bincount(cell.to(torch.int64), minlength=nc).to(torch.int32).cpu().numpy()
        assert np.array_equal(bc, count)
        # ---- sampled particles, followed one by one by the oracle
        k = 4096
        idx = np.sort(rng.choice(n0, size=k, replace=False))
        if margin:
            edge = np.concatenate([np.arange(0, 256), np.arange(n0 - 256, n0)])  # some that do hit a wall
            idx = np.unique(np.concatenate([idx, edge]))
        st = _oracle_subset(inp, s, idx, steps)
        live = st.cell >= 0
        lo = offset[st.cell[live]].astype(np.int64)
        hi = offset[st.cell[live] + 1].astype(np.int64)
        xs, vxs, vys, vzs = (torch.from_numpy(a[live]).to(x.device) for a in (st.x, st.vx, st.vy, st.vz))
        lo_t, hi_t = torch.from_numpy(lo).to(x.device), torch.from_numpy(hi).to(x.device)
        found = torch.zeros(len(lo), dtype=torch.int64, device=x.device)
        width = int((hi - lo).max())
        for j in range(width):
            p = lo_t + j
            ok = p < hi_t
            pc = torch.where(ok, p, lo_t)
            hit = ok & (x[pc] == xs) & (vx[pc] == vxs) & (vy[pc] == vys) & (vz[pc] == vzs)
            found += hit.to(torch.int64)
        assert bool((found == 1).all()), (f"config {config} species {si}: {(found != 1).sum().item()} of {len(lo)} "
                                          f"sampled particles not found bit-exactly in their final cell")
        # ---- exact wall counts: only particles that start within `margin` cells of a wall can reach it
        if inp["boundary"] == workloads.ABSORBING:
            near = np.flatnonzero((s["cell"] < margin) | (s["cell"] >= nc - margin))
            sw = _oracle_subset(inp, s, near, steps)
            dead = sw.cell < 0
            start = s["cell"][near][dead]
            reach = np.minimum(start, nc - 1 - start)
            assert reach.max(initial=0) < margin // 2, "margin too small to certify the wall counts"
            assert (wf["left_total"], wf["right_total"]) == (int(sw.wall[0]), int(sw.wall[1]))
        else:
            assert wf["left_total"] == 0 and wf["right_total"] == 0
    pic.pic_destroy(sim)


# ---- the whole run, element by element (north_star: "arranged order bit-exact ... on all five configs") ----------
@pytest.mark.parametrize("config,single_thread_too", [(2, True), (3, False), (4, False), (5, False)])
def test_fullsize_whole_run_elementwise(config, single_thread_too):
    """Every step of the config at full size, in bench.py's launch configuration, one pic_push_all(nsteps) (as the e2e
    leg; the two species of config 3 overlap on their own streams) -- then the final state against the oracle's: the five arrays bit for bit over [0, n_live),
    counts, offsets, walls.  A wrong rank inside a cell at any step changes the final order, so this covers the
    stable order the sampled test below cannot see."""
    inp = workloads.make(config)
    nc, steps, ae = inp["nc"], inp["steps"], inp["arrange_every"]
    assert steps % ae == 0
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        sim, _ = make_pair(inp, stream=stream)
    del _
    pic.pic_push_all(sim, steps)
    pic.pic_sync(sim)
    for si, (sp, s) in enumerate(zip(sim.species, inp["species"])):
        kw = dict(nc=nc, dx=inp["dx"], dt=inp["dt"], boundary=inp["boundary"], E=inp["E"], qm=s["qm"], B=inp["B"],
                  arrange_every=ae)
        st = oracle.State(s["x"], s["vx"], s["vy"], s["vz"], s["cell"], threads=0, **kw)
        st.push(steps)
        compare(sp, st, where=f"config {config} full size, all {steps} steps, species {si} (threaded oracle)",
                counts=True, nc=nc)
        if single_thread_too:
            st1 = oracle.State(s["x"], s["vx"], s["vy"], s["vz"], s["cell"], **kw)
            st1.push(steps)
            for a, b in zip(st1.live(), st.live()):
                assert np.array_equal(a, b), "threaded oracle differs from the single-thread oracle"
            assert np.array_equal(st1.wall, st.wall) and np.array_equal(st1.offset, st.offset)
        assert pic.pic_arrange_info(sp)[1] == 0, "full-size run fell to the general arranger"
        assert pic.pic_fused_info(sp)["decline_reasons"] == 0, "a fused step declined at full size"
        del st
    pic.pic_destroy(sim)


# ---- beyond the configs: particle arrays larger than 2 GiB (maximum sizes) -----------------------------------------------
def test_arrays_beyond_2_gib_elementwise():
    """280 M electrons on 2.8 M periodic cells (config 4's shape, 2.8 times its size): every fp64 array is 2.24 GB, so a
    byte offset no longer fits 31 bits and a slot index approaches 2^28 -- the sizes where 32-bit address arithmetic
    would first go wrong.  Two fused steps, then (option fused = 0) one step of the split kernels (mover, tile-ranked
    scatter) and the deposition, each compared element by element with the threaded oracle."""
    inp = workloads.make(4, nc=2_800_000)
    s = inp["species"][0]
    n0 = len(s["x"])
    assert n0 * 8 > 2**31
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        desc = pic.make_species(s["x"], s["vx"], s["vy"], s["vz"], s["cell"], qm=s["qm"], arrange_every=1)
    stream.synchronize()
    sim = pic.pic_create(nc=inp["nc"], dx=inp["dx"], dt=inp["dt"], boundary=inp["boundary"], E_nodes=inp["E"], B=inp["B"],
                         species=[desc], stream=stream)
    st = oracle.State(s["x"], s["vx"], s["vy"], s["vz"], s["cell"], nc=inp["nc"], dx=inp["dx"], dt=inp["dt"],
                      boundary=inp["boundary"], E=inp["E"], qm=s["qm"], B=inp["B"], arrange_every=1, threads=0)
    sp = sim.species[0]
    pic.pic_push_all(sim, 2)
    st.push(2)
    compare(sp, st, where="280 M particles, two fused steps", counts=True, nc=inp["nc"])
    info = pic.pic_fused_info(sp)
    assert info["active"] == 1 and info["decline_reasons"] == 0, info
    pic.pic_set_option(sim, "fused", 0)
    pic.pic_push(sp, 1)
    st.push(1)
    compare(sp, st, where="280 M particles, one step of the split kernels", counts=True, nc=inp["nc"])
    assert pic.pic_arrange_info(sp)[1] == 0, "fell to the general arranger"
    rho = pic.pic_deposit(sp, -1.0).cpu().numpy()
    ref = st.deposit(-1.0)
    assert np.all(np.abs(rho - ref) <= 1e-12 * np.maximum(np.abs(ref), 1.0))
    pic.pic_destroy(sim)


# Bounds of the full-size closed cycle: about ten times the largest deviation observed; the
# deviation of a particle array is |a-b| / max(|b|, 0.1).
# observed (config 3 / config 4): rho 2.0e-12 / 2.7e-12, phi 2.2e-11 / 4.6e-11, E 3.7e-13 / 5.6e-14, particles 5.1e-12 / 1.4e-11
FULL_RHO_RTOL, FULL_PHI_RTOL, FULL_E_RTOL, FULL_P_RTOL = 1e-11, 1e-10, 4e-12, 1e-10


# ---- the closed cycle at full size ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("config,cycles", [(3, 20), (4, 10)])
def test_fullsize_closed_cycle_against_the_oracle_loop(config, cycles):
    """pic_cycle at BASELINE.json's full sizes (config 3: e- + D+ between absorbing walls, 2 x 20 M particles, 10^5 nodes;
    config 4: 100 M electrons on a ring of 10^6 nodes with a neutralising background): push + arrange, deposit, two
    filter passes, Poisson, E, the field never leaving the device -- against the same loop of the oracle (threaded
    mover / arranger twin, sequential deposition, binary128 Thomas solve).  The fields agree to rounding (DESIGN.md
    section 12), so the particles agree to the tolerance of the reduced closed-loop test and cells, counts, arranged order
    and wall counters bit for bit."""
    inp = workloads.make(config)
    nc, dx, boundary, passes = inp["nc"], inp["dx"], inp["boundary"], 2
    ppc = len(inp["species"][0]["x"]) / nc
    w = 0.25 / ppc
    weights = [-w if s["qm"] < 0 else w for s in inp["species"]]
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        descs = [pic.make_species(s["x"], s["vx"], s["vy"], s["vz"], s["cell"], qm=s["qm"], arrange_every=1)
                 for s in inp["species"]]
    stream.synchronize()
    sim = pic.pic_create(nc=nc, dx=dx, dt=inp["dt"], boundary=boundary, E_nodes=inp["E"], B=inp["B"], species=descs,
                         stream=stream)
    rho_t, phi_t = pic.pic_cycle(sim, cycles, weights, smooth_passes=passes, want_phi=True)
    states = [oracle.State(s["x"], s["vx"], s["vy"], s["vz"], s["cell"], nc=nc, dx=dx, dt=inp["dt"], boundary=boundary,
                           E=inp["E"].copy(), qm=s["qm"], B=inp["B"], arrange_every=1, threads=0) for s in inp["species"]]
    for _ in range(cycles):
        rho_o = np.zeros(nc + 1)
        for si, st in enumerate(states):
            st.push(1)
            rho_o = rho_o + st.deposit(weights[si])
        _, phi_o, E_o = oracle.field_solve(rho_o, nc, dx, boundary, passes)
        for st in states:
            st.E[:] = E_o
    E = pic.pic_get_field(sim)  # settles the pending cycles
    pmax = max(np.max(np.abs(phi_o)), dx * dx * np.max(np.abs(rho_o)))
    dev_rho = np.max(np.abs(rho_t.cpu().numpy() - rho_o)) / max(np.max(np.abs(rho_o)), w)
    dev_phi = np.max(np.abs(phi_t.cpu().numpy() - phi_o)) / pmax
    dev_E = np.max(np.abs(E - E_o)) / max(np.max(np.abs(E_o)), pmax / dx)
    assert dev_rho <= FULL_RHO_RTOL and dev_phi <= FULL_PHI_RTOL and dev_E <= FULL_E_RTOL, (dev_rho, dev_phi, dev_E)
    dev_p = 0.0
    for si, (sp, st) in enumerate(zip(sim.species, states)):
        compare(sp, st, where=f"config {config} full size, {cycles} closed cycles, species {si}", bitwise=False, counts=True,
                nc=nc, rtol=FULL_P_RTOL, atol=0.1 * FULL_P_RTOL)
        g, o = [t.cpu().numpy() for t in sp.state()], st.live()
        dev_p = max(dev_p, max(float(np.max(np.abs(g[k] - o[k]) / np.maximum(np.abs(o[k]), 0.1))) for k in range(4)))
        assert pic.pic_fused_info(sp)["decline_reasons"] == 0
    print(f"full-size closed cycle, config {config}, {cycles} cycles: observed rho {dev_rho:.3e}, phi {dev_phi:.3e}, "
          f"E {dev_E:.3e}, particles {dev_p:.3e}")
    pic.pic_destroy(sim)
