"""pic_deposit_static, the charge deposition for callers that must not allocate device memory.

Some users of libpic cannot let a call allocate: a host code that maps all of its device arrays once at start-up and
keeps them for the run may have no memory left to give, and inside a time loop a hidden cudaMalloc or
cudaFree serialises the whole device and stalls the other streams.  pic_deposit takes its per-cell scratch from the
library's pool, and needs a handle that pic_create allocates; pic_deposit_static takes raw device arrays and keeps the
scratch in a 16 MiB array that is part of libpic.so (PIC_DEPOSIT_STATIC_MAX_NC = 2^20 cells).

The GPU test compares it with the existing path, pic_deposit, on the same arranged state, at the tolerance the
deposition tests use (1e-12 of max(|rho_j|, |weight|)), for two calls in a row that share the scratch array: a large
grid first, then a smaller one with the other boundary type, so the second call runs over whatever the first left
behind.  It also checks that the device's free memory does not move across a call.  The file is named to be collected
last: under `pytest -x` a failure here hides no other test.  It passes alone in a fresh process (the first call does
the per-device set-up) and after the rest of the suite.
"""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_2603_24508_b200 as pic
from paper_2603_24508_b200 import workloads

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
DEP_RTOL = 1e-12  # as tests/test_gpu_parity.py: DEP_RTOL


def test_limit_in_header_and_binding_agree():
    src = open(os.path.join(ROOT, "include", "pic.h")).read()
    m = re.search(r"#define\s+PIC_DEPOSIT_STATIC_MAX_NC\s+\(1\s*<<\s*(\d+)\)", src)
    assert m, "include/pic.h must state the limit"
    assert pic.PIC_DEPOSIT_STATIC_MAX_NC == 1 << int(m.group(1)) == 1 << 20


def test_arguments_are_rejected_before_any_cuda_call():
    """Runs without a GPU: the size and argument checks come first and say why."""
    L = pic.lib()
    buf = (C.c_double * 4)()
    p = C.cast(buf, C.c_void_p)
    too_many = pic.PIC_DEPOSIT_STATIC_MAX_NC + 1
    assert L.pic_deposit_static(p, p, 0, too_many, 1.0, 0, 1.0, 0, p, None) == pic.PIC_ECAPACITY
    msg = pic.pic_last_error()
    assert str(too_many) in msg and str(pic.PIC_DEPOSIT_STATIC_MAX_NC) in msg
    assert L.pic_deposit_static(None, p, 0, 8, 1.0, 0, 1.0, 0, p, None) == pic.PIC_EINVAL
    assert L.pic_deposit_static(p, None, 0, 8, 1.0, 0, 1.0, 0, p, None) == pic.PIC_EINVAL
    assert L.pic_deposit_static(p, p, 0, 8, 1.0, 0, 1.0, 0, None, None) == pic.PIC_EINVAL
    assert L.pic_deposit_static(p, p, -1, 8, 1.0, 0, 1.0, 0, p, None) == pic.PIC_EINVAL
    assert L.pic_deposit_static(p, p, 0, 0, 1.0, 0, 1.0, 0, p, None) == pic.PIC_EINVAL
    assert L.pic_deposit_static(p, p, 0, 8, 0.0, 0, 1.0, 0, p, None) == pic.PIC_EINVAL
    assert L.pic_deposit_static(p, p, 0, 8, 1.0, 0, float("nan"), 0, p, None) == pic.PIC_EINVAL
    assert L.pic_deposit_static(p, p, 0, 8, 1.0, 7, 1.0, 0, p, None) == pic.PIC_EINVAL


def _arranged_case(config, nc, steps):
    """A sim of one reduced config pushed `steps` arranging steps, its existing-path rho for two weights, and the raw
    device arrays a handle-free caller would own: x of the active buffer and the offset table, uploaded."""
    import torch
    inp = workloads.make(config, nc=nc)
    descs = [pic.make_species(s["x"], s["vx"], s["vy"], s["vz"], s["cell"], qm=s["qm"], arrange_every=1)
             for s in inp["species"]]
    sim = pic.pic_create(nc=inp["nc"], dx=inp["dx"], dt=inp["dt"], boundary=inp["boundary"], E_nodes=inp["E"],
                         B=inp["B"], species=descs)
    sp = sim.species[0]
    pic.pic_push(sp, steps)
    x = sp.state()[0]  # syncs; slots [0, n_live) of the active buffer
    _, off = pic.pic_cell_counts(sp, nc)
    assert off[nc] == x.numel()
    offset = torch.from_numpy(off).cuda()
    return sim, sp, inp, x, offset


def _close(got, ref, weight, where):
    scale = np.maximum(np.abs(ref), abs(weight))
    err = np.abs(got - ref) / scale
    assert np.all(err <= DEP_RTOL), f"{where}: differs from pic_deposit, max {err.max():.3e} at node {err.argmax()}"


@pytest.mark.gpu
def test_static_scratch_deposit_matches_pic_deposit_on_two_calls_in_a_row():
    import torch
    # first state: absorbing walls, 40,000 cells, some particles already absorbed (n < the initial count)
    simA, spA, inpA, xA, offA = _arranged_case(2, 40_000, 12)
    # second state: periodic ring, far fewer cells: its call runs over the first call's left-overs in the scratch
    simB, spB, inpB, xB, offB = _arranged_case(1, 1_024, 5)
    refA = pic.pic_deposit(spA, -0.75).cpu().numpy()
    refB1 = pic.pic_deposit(spB, 1.5)
    refB = pic.pic_deposit(spB, 0.25, rho=refB1, accumulate=True).cpu().numpy()  # accumulate, as a second species would
    rhoA = torch.full((inpA["nc"] + 1,), 7.0, dtype=torch.float64, device="cuda")  # overwritten, not added to
    rhoB = torch.full((inpB["nc"] + 1,), -3.0, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()

    # two calls in a row on one stream, nothing between them
    pic.pic_deposit_static(xA, offA, nc=inpA["nc"], dx=inpA["dx"], boundary=inpA["boundary"], weight=-0.75, rho=rhoA)
    pic.pic_deposit_static(xB, offB, nc=inpB["nc"], dx=inpB["dx"], boundary=inpB["boundary"], weight=1.5, rho=rhoB)
    torch.cuda.synchronize()
    _close(rhoA.cpu().numpy(), refA, 0.75, "first call (absorbing, 40,000 cells)")
    gotB1 = rhoB.cpu().numpy()

    # a third, accumulating call; the device's free memory must not move across it (set-up was done by the first call)
    free0, _ = torch.cuda.mem_get_info()
    pic.pic_deposit_static(xB, offB, nc=inpB["nc"], dx=inpB["dx"], boundary=inpB["boundary"], weight=0.25, rho=rhoB,
                           accumulate=True)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, f"free device memory moved by {free0 - free1} bytes across pic_deposit_static"
    _close(rhoB.cpu().numpy(), refB, 1.5, "second + accumulating call (periodic, 1,024 cells)")
    assert gotB1[0] == gotB1[-1], "periodic grid: nodes 0 and nc are one point"
    # on the ring no particle is ever absorbed, pic_deposit's bound on n is n itself: same lanes per cell, same tree, same bits
    assert np.array_equal(gotB1, pic.pic_deposit(spB, 1.5).cpu().numpy())

    # the first case once more after the small one: still right, and bit-identical to its first run
    again = torch.empty_like(rhoA)
    pic.pic_deposit_static(xA, offA, nc=inpA["nc"], dx=inpA["dx"], boundary=inpA["boundary"], weight=-0.75, rho=again)
    torch.cuda.synchronize()
    assert torch.equal(again, rhoA)

    # beyond the limit: refused with both numbers in the message, nothing launched, rho untouched
    with pytest.raises(pic.PicError) as e:
        pic.pic_deposit_static(xB, torch.zeros(pic.PIC_DEPOSIT_STATIC_MAX_NC + 2, dtype=torch.int32, device="cuda"),
                               nc=pic.PIC_DEPOSIT_STATIC_MAX_NC + 1, dx=1.0, boundary=0, weight=1.0,
                               rho=torch.zeros(pic.PIC_DEPOSIT_STATIC_MAX_NC + 2, dtype=torch.float64, device="cuda"))
    assert e.value.status == pic.PIC_ECAPACITY and str(pic.PIC_DEPOSIT_STATIC_MAX_NC) in str(e.value)
    pic.pic_sync(simA)
    pic.pic_sync(simB)
