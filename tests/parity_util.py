"""Shared driver of the GPU parity tests: runs libpic (through the Python binding of the C ABI)
and the CPU oracle from the same seeded inputs and compares them element by element.

The bar (BASELINE.json north_star): x, vx, vy, vz within
|a-b| <= max(1e-14, 1e-12*|b|); cell indices, dead flags, per-cell counts, offsets, arranged
order, slot counts and wall counters bit-exact.  Because a cell index is decided by
floor(x/dx), both sides execute the same sequence of individually rounded binary64 operations
and the floating-point arrays are in fact expected to agree bitwise; `bitwise=True` asserts it.
"""
import numpy as np

import oracle
import paper_2603_24508_b200 as pic

RTOL, ATOL = 1e-12, 1e-14


def close(a, b, rtol=RTOL, atol=ATOL):
    return np.all(np.abs(a - b) <= np.maximum(atol, rtol * np.abs(b)))


def make_pair(inp, *, arrange_every=None, capacity_pad=0, workspace=True, options=None, stream=None):
    """-> (sim, [oracle.State per species])"""
    ae = inp["arrange_every"] if arrange_every is None else arrange_every
    states, descs = [], []
    for s in inp["species"]:
        states.append(oracle.State(s["x"], s["vx"], s["vy"], s["vz"], s["cell"], nc=inp["nc"], dx=inp["dx"],
                                   dt=inp["dt"], boundary=inp["boundary"], E=inp["E"], qm=s["qm"], B=inp["B"],
                                   arrange_every=ae))
        descs.append(pic.make_species(s["x"], s["vx"], s["vy"], s["vz"], s["cell"], qm=s["qm"], arrange_every=ae,
                                      capacity=len(s["x"]) + capacity_pad, workspace=workspace))
    sim = pic.pic_create(nc=inp["nc"], dx=inp["dx"], dt=inp["dt"], boundary=inp["boundary"], E_nodes=inp["E"],
                         B=inp["B"], species=descs, stream=stream)
    for k, v in (options or {}).items():
        pic.pic_set_option(sim, k, v)
    return sim, states


def compare(sp, st, *, where="", bitwise=True, counts=False, nc=None, rtol=RTOL, atol=ATOL):
    """Compare the GPU species `sp` with the oracle state `st` over the slots in use."""
    n_gpu = pic.pic_n_slots(sp)
    assert n_gpu == st.n, f"{where}: slots in use {n_gpu} != oracle {st.n}"
    g = [t.cpu().numpy() for t in sp.state()]
    o = st.live()
    names = ("x", "vx", "vy", "vz", "cell")
    assert np.array_equal(g[4], o[4]), f"{where}: cell / dead flags differ at {np.flatnonzero(g[4] != o[4])[:8]}"
    for k in range(4):
        assert close(g[k], o[k], rtol, atol), f"{where}: {names[k]} outside tolerance, max abs diff {np.max(np.abs(g[k] - o[k]))}"
        if bitwise:
            assert np.array_equal(g[k], o[k]), (f"{where}: {names[k]} not bitwise equal at "
                                                f"{np.flatnonzero(g[k] != o[k])[:8]}")
    wf = pic.pic_wall_flux(sp)
    assert wf["left_total"] == int(st.wall[0]) and wf["right_total"] == int(st.wall[1]), \
        f"{where}: wall counters {wf} != oracle {st.wall}"
    assert wf["steps_total"] == st.steps
    if counts:
        c, off = pic.pic_cell_counts(sp, nc)
        assert np.array_equal(c, st.count), f"{where}: per-cell counts differ"
        assert np.array_equal(off, st.offset), f"{where}: offsets differ"
    return wf


def run_stepwise(inp, steps, *, arrange_every=None, options=None, bitwise=True, check_every=1):
    """Drive both sides one step per call, comparing after every `check_every` steps."""
    sim, states = make_pair(inp, arrange_every=arrange_every, options=options)
    ae = inp["arrange_every"] if arrange_every is None else arrange_every
    for step in range(1, steps + 1):
        for sp, st in zip(sim.species, states):
            pic.pic_push(sp, 1)
            st.push(1)
        if step % check_every == 0 or step == steps:
            for si, (sp, st) in enumerate(zip(sim.species, states)):
                arranged = ae > 0 and step % ae == 0
                compare(sp, st, where=f"step {step} species {si}", bitwise=bitwise, counts=arranged, nc=inp["nc"])
    pic.pic_sync(sim)
    return sim, states


def run_bulk(inp, steps, *, arrange_every=None, options=None, bitwise=True):
    """One pic_push(sp, steps) call against steps oracle steps; final state compared."""
    sim, states = make_pair(inp, arrange_every=arrange_every, options=options)
    ae = inp["arrange_every"] if arrange_every is None else arrange_every
    for si, (sp, st) in enumerate(zip(sim.species, states)):
        pic.pic_push(sp, steps)
        st.push(steps)
        compare(sp, st, where=f"bulk {steps} species {si}", bitwise=bitwise, counts=ae > 0 and steps % ae == 0,
                nc=inp["nc"])
    pic.pic_sync(sim)
    return sim, states
