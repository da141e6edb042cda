"""paper_2603_24508_b200 -- Python binding of libpic (include/pic.h): the BIT1-style particle
mover + arranger of arxiv/paper_2603_24508 on one B200.

Argument marshalling only: every step of the path runs in the CUDA kernels of csrc/ behind the
C ABI; torch supplies device memory and streams.  The functions carry the C names
(pic_create, pic_push, pic_arrange, pic_wall_flux, ...).  There is no CPU fallback: if
libpic.so has not been built (python -m paper_2603_24508_b200.build) loading fails loudly.
"""
import ctypes as C
import os

import numpy as np

PIC_OK, PIC_EINVAL, PIC_ENOMEM, PIC_ECUDA, PIC_ECAPACITY, PIC_ESTATE = 0, -1, -2, -3, -4, -5
PIC_PERIODIC, PIC_ABSORBING = 0, 1

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpic.so")

EXPORTS = [
    "pic_create", "pic_species_at", "pic_push", "pic_arrange", "pic_wall_flux", "pic_set_field", "pic_n_slots",
    "pic_active_buffer", "pic_cell_counts", "pic_step_count", "pic_arrange_info", "pic_workspace_bytes",
    "pic_set_option", "pic_launch_count", "pic_sync", "pic_destroy", "pic_strerror", "pic_last_error",
    "pic_run_host", "pic_kernel_time", "pic_fused_info", "pic_deposit", "pic_n_live", "pic_set_field_device",
    "pic_solve_field", "pic_get_field", "pic_push_all", "pic_trim_memory", "pic_cycle", "pic_deposit_static",
]
PIC_DEPOSIT_STATIC_MAX_NC = 1 << 20  # include/pic.h: cells the built-in scratch array of pic_deposit_static holds


class PicError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        msg = f"{where}: {pic_strerror(status)} ({status})"
        extra = pic_last_error()
        if status in (PIC_ECUDA, PIC_ESTATE) and extra:
            msg += f": {extra}"
        super().__init__(msg)


class pic_grid_desc(C.Structure):
    _fields_ = [("nc", C.c_int32), ("boundary", C.c_int32), ("dx", C.c_double), ("dt", C.c_double),
                ("E_nodes", C.POINTER(C.c_double)), ("B", C.c_double * 3), ("stream", C.c_void_p)]


class pic_species_desc(C.Structure):
    _fields_ = [("qm", C.c_double), ("n", C.c_int64), ("capacity", C.c_int64),
                ("x", C.c_void_p * 2), ("vx", C.c_void_p * 2), ("vy", C.c_void_p * 2), ("vz", C.c_void_p * 2),
                ("cell", C.c_void_p * 2), ("arrange_every", C.c_int32), ("reserved", C.c_int32),
                ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t)]


class pic_wall_flux_t(C.Structure):
    _fields_ = [("left_total", C.c_uint64), ("right_total", C.c_uint64), ("left_recent", C.c_uint64),
                ("right_recent", C.c_uint64), ("steps_total", C.c_uint64), ("steps_recent", C.c_uint64)]


class pic_host_species(C.Structure):
    _fields_ = [("qm", C.c_double), ("n", C.c_int64),
                ("x", C.c_void_p), ("vx", C.c_void_p), ("vy", C.c_void_p), ("vz", C.c_void_p), ("cell", C.c_void_p),
                ("arrange_every", C.c_int32), ("reserved", C.c_int32),
                ("n_out", C.c_int64), ("wall_left", C.c_uint64), ("wall_right", C.c_uint64)]


_lib = None


def lib():
    """The loaded libpic.so; raises if it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2603_24508_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i32p, i64p = C.c_void_p, C.POINTER(C.c_int32), C.POINTER(C.c_int64)
        L.pic_create.argtypes = [C.POINTER(pic_grid_desc), C.POINTER(pic_species_desc), C.c_int, C.POINTER(vp)]
        L.pic_species_at.argtypes = [vp, C.c_int]
        L.pic_species_at.restype = vp
        L.pic_push.argtypes = [vp, C.c_int]
        L.pic_push_all.argtypes = [vp, C.c_int]
        L.pic_arrange.argtypes = [vp]
        L.pic_wall_flux.argtypes = [vp, C.POINTER(pic_wall_flux_t)]
        L.pic_set_field.argtypes = [vp, C.POINTER(C.c_double)]
        L.pic_n_slots.argtypes = [vp, i64p]
        L.pic_n_live.argtypes = [vp, i64p]
        L.pic_set_field_device.argtypes = [vp, vp]
        L.pic_solve_field.argtypes = [vp, vp, C.c_int, vp]
        L.pic_get_field.argtypes = [vp, C.POINTER(C.c_double)]
        L.pic_active_buffer.argtypes = [vp, C.POINTER(C.c_int)]
        L.pic_cell_counts.argtypes = [vp, i32p, i32p]
        L.pic_step_count.argtypes = [vp, i64p]
        L.pic_arrange_info.argtypes = [vp, i32p, i32p]
        L.pic_workspace_bytes.argtypes = [C.c_int32, C.c_int64]
        L.pic_workspace_bytes.restype = C.c_size_t
        L.pic_set_option.argtypes = [vp, C.c_char_p, C.c_int]
        L.pic_launch_count.argtypes = [vp, C.POINTER(C.c_uint64)]
        L.pic_kernel_time.argtypes = [vp, C.c_char_p, C.POINTER(C.c_double), C.POINTER(C.c_uint64)]
        L.pic_fused_info.argtypes = [vp, i32p, i32p, i32p, i32p]
        L.pic_deposit.argtypes = [vp, C.c_double, vp, C.c_int]
        L.pic_deposit_static.argtypes = [vp, vp, C.c_int64, C.c_int32, C.c_double, C.c_int32, C.c_double, C.c_int, vp, vp]
        L.pic_sync.argtypes = [vp]
        L.pic_destroy.argtypes = [vp]
        L.pic_destroy.restype = None
        L.pic_strerror.argtypes = [C.c_int]
        L.pic_strerror.restype = C.c_char_p
        L.pic_last_error.argtypes = []
        L.pic_last_error.restype = C.c_char_p
        L.pic_trim_memory.argtypes = []
        L.pic_cycle.argtypes = [vp, C.c_int, C.POINTER(C.c_double), C.c_int, vp, vp]
        L.pic_run_host.argtypes = [C.POINTER(pic_grid_desc), C.POINTER(pic_host_species), C.c_int, C.c_int]
        _lib = L
    return _lib


def pic_strerror(status):
    return lib().pic_strerror(int(status)).decode()


def pic_last_error():
    return lib().pic_last_error().decode()


def _check(rc, where):
    if rc != PIC_OK:
        raise PicError(rc, where)


def pic_workspace_bytes(nc, capacity):
    return int(lib().pic_workspace_bytes(int(nc), int(capacity)))


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class Species:
    """Handle of one species (pic_species*) plus the torch tensors it lives in."""

    def __init__(self, sim, handle, bufs, workspace):
        self.sim, self.handle, self.bufs, self.workspace = sim, handle, bufs, workspace

    def state(self):
        """(x, vx, vy, vz, cell) torch tensors of the active buffer set, sliced to the slots in use."""
        n = pic_n_slots(self)
        b = pic_active_buffer(self)
        return tuple(t[:n] for t in self.bufs[b])


class Sim:
    """Handle of a simulation (pic_sim*)."""

    def __init__(self, handle, species, keep, nc=None, stream=None):
        self.handle, self.species, self._keep, self.nc, self.stream = handle, species, keep, nc, stream

    def __del__(self):
        try:
            pic_destroy(self)
        except Exception:
            pass


def make_species(x, vx, vy, vz, cell, *, qm, arrange_every=0, capacity=None, workspace=True, device="cuda"):
    """Marshalling helper: upload host arrays (numpy) into two torch buffer sets of `capacity`
    slots and describe them for pic_create.  workspace=True allocates pic_workspace_bytes."""
    import torch
    n = len(x)
    cap = int(capacity if capacity is not None else n)
    cap_alloc = max(cap, 1)
    bufs = []
    for b in range(2):
        fs = [torch.empty(cap_alloc, dtype=torch.float64, device=device) for _ in range(4)]
        fs.append(torch.empty(cap_alloc, dtype=torch.int32, device=device))
        bufs.append(fs)
    if n:
        for t, a in zip(bufs[0], (x, vx, vy, vz, cell)):
            t[:n].copy_(torch.from_numpy(np.ascontiguousarray(a)))
    return {"qm": float(qm), "n": n, "capacity": cap, "bufs": bufs, "arrange_every": int(arrange_every),
            "workspace": workspace}


def pic_create(*, nc, dx, dt, boundary, E_nodes, B, species, stream=None):
    """pic_create(grid, species): species is a list of make_species(...) dicts.  Returns Sim."""
    import torch
    E = np.ascontiguousarray(E_nodes, dtype=np.float64)
    if E.shape != (nc + 1,):
        raise ValueError("E_nodes must have nc+1 entries")
    g = pic_grid_desc()
    g.nc, g.boundary, g.dx, g.dt = int(nc), int(boundary), float(dx), float(dt)
    g.E_nodes = _dptr(E)
    g.B = (C.c_double * 3)(*[float(b) for b in B])
    if stream is None:
        stream = torch.cuda.current_stream()
    g.stream = C.c_void_p(stream.cuda_stream)
    descs = (pic_species_desc * len(species))()
    keep = [E, stream]
    wss = []
    for d, s in zip(descs, species):
        d.qm, d.n, d.capacity = s["qm"], s["n"], s["capacity"]
        for b in range(2):
            fx, fvx, fvy, fvz, fc = s["bufs"][b]
            d.x[b], d.vx[b], d.vy[b], d.vz[b], d.cell[b] = (fx.data_ptr(), fvx.data_ptr(), fvy.data_ptr(),
                                                           fvz.data_ptr(), fc.data_ptr())
        d.arrange_every = s["arrange_every"]
        ws = s.get("workspace")
        if ws is True:
            ws = torch.empty(pic_workspace_bytes(nc, s["capacity"]), dtype=torch.uint8, device=s["bufs"][0][0].device)
        if ws is None or ws is False:
            d.workspace, d.workspace_bytes = None, 0
            ws = None
        else:
            d.workspace, d.workspace_bytes = ws.data_ptr(), ws.numel() * ws.element_size()
        wss.append(ws)
        keep.append(s["bufs"])
    torch.cuda.current_stream().synchronize()  # uploads in make_species ran on torch's current stream
    h = C.c_void_p()
    _check(lib().pic_create(C.byref(g), descs, len(species), C.byref(h)), "pic_create")
    sim = Sim(h, [], keep, nc=int(nc), stream=stream)
    for i, s in enumerate(species):
        sim.species.append(Species(sim, C.c_void_p(lib().pic_species_at(h, i)), s["bufs"], wss[i]))
    return sim


def pic_species_at(sim, i):
    return sim.species[i]


def pic_push(sp, nsteps=1):
    _check(lib().pic_push(sp.handle, int(nsteps)), "pic_push")


def pic_trim_memory():
    """Return the device memory cached by the library's pool (freed handles, pic_run_host arenas) to the driver."""
    _check(lib().pic_trim_memory(), "pic_trim_memory")


def pic_push_all(sim, nsteps=1):
    """Every species of the sim, nsteps steps each; the species' kernels overlap on internal streams."""
    _check(lib().pic_push_all(sim.handle, int(nsteps)), "pic_push_all")


def pic_arrange(sp):
    _check(lib().pic_arrange(sp.handle), "pic_arrange")


def pic_wall_flux(sp):
    out = pic_wall_flux_t()
    _check(lib().pic_wall_flux(sp.handle, C.byref(out)), "pic_wall_flux")
    return {k: int(getattr(out, k)) for k, _ in pic_wall_flux_t._fields_}


def pic_set_field(sim, E_nodes):
    E = np.ascontiguousarray(E_nodes, dtype=np.float64)
    _check(lib().pic_set_field(sim.handle, _dptr(E)), "pic_set_field")


def pic_set_field_device(sim, E_dev):
    """pic_set_field_device: E (torch float64 device tensor, nc+1) copied on the sim's stream; no host round trip."""
    import torch
    assert E_dev.dtype == torch.float64 and E_dev.numel() == sim.nc + 1 and E_dev.is_contiguous() and E_dev.is_cuda
    sim.stream.wait_stream(torch.cuda.current_stream())  # E_dev was produced on torch's current stream
    _check(lib().pic_set_field_device(sim.handle, C.c_void_p(E_dev.data_ptr())), "pic_set_field_device")
    torch.cuda.current_stream().wait_stream(sim.stream)  # the caller may overwrite E_dev afterwards


def pic_solve_field(sim, rho, smooth_passes=0, phi=None, want_phi=False):
    """pic_solve_field: smooth -> Poisson -> E on the device; E replaces the sim's field.  rho: torch float64 device
    tensor (nc+1), as pic_deposit returns it.  Returns phi (device tensor) if want_phi or phi is given, else None."""
    import torch
    assert rho.dtype == torch.float64 and rho.numel() == sim.nc + 1 and rho.is_contiguous() and rho.is_cuda
    if phi is None and want_phi:
        phi = torch.empty(sim.nc + 1, dtype=torch.float64, device=rho.device)
    if phi is not None:
        assert phi.dtype == torch.float64 and phi.numel() == sim.nc + 1 and phi.is_contiguous()
    sim.stream.wait_stream(torch.cuda.current_stream())
    _check(lib().pic_solve_field(sim.handle, C.c_void_p(rho.data_ptr()), int(smooth_passes),
                                 C.c_void_p(phi.data_ptr()) if phi is not None else None), "pic_solve_field")
    torch.cuda.current_stream().wait_stream(sim.stream)
    return phi


def pic_cycle(sim, ncycles, weights, smooth_passes=0, rho=None, phi=None, want_phi=False):
    """pic_cycle: ncycles closed PIC cycles (push all species, deposit, smooth + Poisson + E) enqueued without a host
    round trip.  weights: one per species.  rho / phi: torch float64 device tensors (nc+1), allocated if None (phi only
    when want_phi); they are kept alive by the Sim until the next call.  Returns (rho, phi)."""
    import torch
    dev = sim.species[0].bufs[0][0].device
    if rho is None:
        rho = torch.empty(sim.nc + 1, dtype=torch.float64, device=dev)
    if phi is None and want_phi:
        phi = torch.empty(sim.nc + 1, dtype=torch.float64, device=dev)
    for t in (rho, phi):
        if t is not None:
            assert t.dtype == torch.float64 and t.numel() == sim.nc + 1 and t.is_contiguous() and t.is_cuda
    w = (C.c_double * len(sim.species))(*[float(x) for x in weights])
    assert len(weights) == len(sim.species)
    # The library keeps the rho / phi pointers of EVERY call whose cycles are still unchecked and, should a fused step
    # have declined, writes into all of them at its next synchronising call: hold every pair until then (a caller who
    # drops the returned rho must not hand its memory back to torch's allocator under the library's feet).
    keep = sim.__dict__.setdefault("_cycle_keep", [])
    if len(keep) >= 64:  # bound the list: settle what is pending (pic_sync clears it)
        pic_sync(sim)
    if not any(r is rho and p is phi for r, p in keep):
        keep.append((rho, phi))
    sim.stream.wait_stream(torch.cuda.current_stream())
    _check(lib().pic_cycle(sim.handle, int(ncycles), w, int(smooth_passes), C.c_void_p(rho.data_ptr()),
                           C.c_void_p(phi.data_ptr()) if phi is not None else None), "pic_cycle")
    torch.cuda.current_stream().wait_stream(sim.stream)
    return rho, phi


def pic_get_field(sim):
    """pic_get_field -> numpy array of the nc+1 node values of E in force."""
    E = np.empty(sim.nc + 1, dtype=np.float64)
    _check(lib().pic_get_field(sim.handle, _dptr(E)), "pic_get_field")
    return E


def pic_n_live(sp):
    n = C.c_int64()
    _check(lib().pic_n_live(sp.handle, C.byref(n)), "pic_n_live")
    return n.value


def pic_n_slots(sp):
    n = C.c_int64()
    _check(lib().pic_n_slots(sp.handle, C.byref(n)), "pic_n_slots")
    return n.value


def pic_active_buffer(sp):
    w = C.c_int()
    _check(lib().pic_active_buffer(sp.handle, C.byref(w)), "pic_active_buffer")
    return w.value


def pic_cell_counts(sp, nc):
    count = np.empty(nc, dtype=np.int32)
    offset = np.empty(nc + 1, dtype=np.int32)
    _check(lib().pic_cell_counts(sp.handle, count.ctypes.data_as(C.POINTER(C.c_int32)),
                                 offset.ctypes.data_as(C.POINTER(C.c_int32))), "pic_cell_counts")
    return count, offset


def pic_step_count(sp):
    n = C.c_int64()
    _check(lib().pic_step_count(sp.handle, C.byref(n)), "pic_step_count")
    return n.value


def pic_arrange_info(sp):
    w, g = C.c_int32(), C.c_int32()
    _check(lib().pic_arrange_info(sp.handle, C.byref(w), C.byref(g)), "pic_arrange_info")
    return w.value, g.value


def pic_deposit(sp, weight, rho=None, accumulate=False):
    """pic_deposit: charge density on the nc+1 nodes (torch float64 device tensor; allocated if None)."""
    import torch
    nc = sp.sim.nc
    if rho is None:
        rho = torch.zeros(nc + 1, dtype=torch.float64, device=sp.bufs[0][0].device)
    sp.sim.stream.wait_stream(torch.cuda.current_stream())
    assert rho.dtype == torch.float64 and rho.numel() == nc + 1 and rho.is_contiguous()
    _check(lib().pic_deposit(sp.handle, float(weight), C.c_void_p(rho.data_ptr()), 1 if accumulate else 0), "pic_deposit")
    torch.cuda.current_stream().wait_stream(sp.sim.stream)  # rho is produced on the sim's stream
    return rho


def pic_deposit_static(x, offset, *, nc, dx, boundary, weight, rho, accumulate=False, stream=None):
    """pic_deposit_static: pic_deposit without a handle and without any device allocation, for a caller whose time
    loop must not allocate (all device memory handed out at start-up, or an allocation would stall its other streams;
    include/pic.h has the full reasoning).  Every array is the caller's: x (float64, the n arranged positions), offset
    (int32, nc+1, offset[nc] = n), rho (float64, nc+1, the output) are CUDA tensors; the binding creates none and the
    library uses a 16 MiB array built into libpic.so as scratch, so nc <= PIC_DEPOSIT_STATIC_MAX_NC (PicError with
    PIC_ECAPACITY beyond it).  Runs on `stream` (default: torch's current stream).  All calls on a device share that
    one scratch array: keep them on one stream, overlapping calls race.  The first call on a device also looks up the
    array's device address; make it during set-up."""
    import torch
    assert x.is_cuda and x.dtype == torch.float64 and x.is_contiguous() and x.dim() == 1
    assert offset.is_cuda and offset.dtype == torch.int32 and offset.is_contiguous() and offset.numel() == nc + 1
    assert rho.is_cuda and rho.dtype == torch.float64 and rho.is_contiguous() and rho.numel() == nc + 1
    st = stream if stream is not None else torch.cuda.current_stream()
    rc = lib().pic_deposit_static(C.c_void_p(x.data_ptr()), C.c_void_p(offset.data_ptr()), int(x.numel()), int(nc),
                                  float(dx), int(boundary), float(weight), 1 if accumulate else 0,
                                  C.c_void_p(rho.data_ptr()), C.c_void_p(st.cuda_stream))
    if rc != PIC_OK:
        err = PicError(rc, "pic_deposit_static")
        if rc in (PIC_EINVAL, PIC_ECAPACITY):  # this call always leaves the reason in pic_last_error
            err.args = (f"{err.args[0]}: {pic_last_error()}",)
        raise err
    return rho


def pic_fused_info(sp):
    """-> dict(active, decline_reasons, stage_slots, ctas_per_sm) of the fused push+arrange step."""
    v = [C.c_int32() for _ in range(4)]
    _check(lib().pic_fused_info(sp.handle, *[C.byref(x) for x in v]), "pic_fused_info")
    return dict(zip(("active", "decline_reasons", "stage_slots", "ctas_per_sm"), (x.value for x in v)))


def pic_set_option(sim, key, value):
    _check(lib().pic_set_option(sim.handle, key.encode(), int(value)), "pic_set_option")


def pic_launch_count(sim):
    n = C.c_uint64()
    _check(lib().pic_launch_count(sim.handle, C.byref(n)), "pic_launch_count")
    return n.value


def pic_kernel_time(sim, kernel):
    """-> (milliseconds, timed launches) of one kernel class since the previous query (option kernel_timing)."""
    ms, n = C.c_double(), C.c_uint64()
    _check(lib().pic_kernel_time(sim.handle, kernel.encode(), C.byref(ms), C.byref(n)), "pic_kernel_time")
    return ms.value, n.value


def pic_sync(sim):
    _check(lib().pic_sync(sim.handle), "pic_sync")
    keep = sim.__dict__.get("_cycle_keep")
    if keep:  # pending cycles are settled: only the latest pair may still be in the caller's hands
        del keep[:-1]


def pic_destroy(sim):
    if sim.handle:
        lib().pic_destroy(sim.handle)
        sim.handle = None


def pic_run_host(*, nc, dx, dt, boundary, E_nodes, B, species, nsteps, stream=None):
    """pic_run_host: end-to-end call with HOST buffers.  species: list of dicts with qm,
    arrays=[x, vx, vy, vz, cell] (numpy arrays or pinned CPU torch tensors, overwritten with the
    final state) and arrange_every.  Returns [(n_out, wall_left, wall_right), ...]."""
    E = np.ascontiguousarray(E_nodes, dtype=np.float64)
    g = pic_grid_desc()
    g.nc, g.boundary, g.dx, g.dt = int(nc), int(boundary), float(dx), float(dt)
    g.E_nodes = _dptr(E)
    g.B = (C.c_double * 3)(*[float(b) for b in B])
    g.stream = C.c_void_p(stream.cuda_stream if stream is not None else 0)
    hs = (pic_host_species * len(species))()
    for h, s in zip(hs, species):
        a = s["arrays"]
        if len(a) != 5:
            raise ValueError("arrays must be [x, vx, vy, vz, cell]")
        for k, t in enumerate(a):  # the C side reads and overwrites n elements of each: check before handing pointers over
            want = "int32" if k == 4 else "float64"
            if hasattr(t, "data_ptr"):
                ok = str(t.dtype).endswith(want) and t.is_contiguous() and not t.is_cuda and t.dim() == 1
            else:
                ok = isinstance(t, np.ndarray) and t.dtype == np.dtype(want) and t.flags.c_contiguous and t.ndim == 1 \
                    and t.flags.writeable
            if not ok:
                raise ValueError(f"arrays[{k}] must be a contiguous, writable, 1-D host {want} array")
            if len(t) != len(a[0]):
                raise ValueError("the five arrays of a species must have equal lengths")
        ptrs = [t.data_ptr() if hasattr(t, "data_ptr") else t.ctypes.data for t in a]
        h.qm, h.n = float(s["qm"]), len(a[0])
        h.x, h.vx, h.vy, h.vz, h.cell = ptrs
        h.arrange_every = int(s.get("arrange_every", 0))
    _check(lib().pic_run_host(C.byref(g), hs, len(species), int(nsteps)), "pic_run_host")
    return [(int(h.n_out), int(h.wall_left), int(h.wall_right)) for h in hs]
