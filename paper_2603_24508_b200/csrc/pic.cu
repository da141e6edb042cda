// pic.cu -- host side of libpic: the C ABI of include/pic.h (handles, validation, per-species
// constants, kernel launches on the caller's stream).  No torch types; no CPU compute path.
#include "../../include/pic.h"

#include <chrono>
#include <climits>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include <nvtx3/nvToolsExt.h> // header-only; a no-op unless a profiler (nsys, ncu --nvtx) is attached

#include "pic_device.cuh"
#include "mover.cuh"
#include "scan.cuh"
#include "arranger.cuh"
#include "general.cuh"
#include "tilesort.cuh"
#include "deposit.cuh"
#include "field.cuh"
#include "fused.cuh"

using namespace pic;

static thread_local char g_err[512] = "";

static int cuda_fail(cudaError_t e, const char *what)
{
    snprintf(g_err, sizeof g_err, "%s: %s", what, cudaGetErrorString(e));
    return PIC_ECUDA;
}
#define CU(call)                                            \
    do {                                                    \
        cudaError_t e_ = (call);                            \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call); \
    } while (0)

enum { K_MOVER = 0, K_HIST, K_SCAN, K_SCATTER, K_GENERAL, K_FUSED, K_DEPOSIT, K_FIELD, K_COUNT };
static const char *const K_NAMES[K_COUNT] = {"mover", "hist", "scan", "scatter", "general", "fused", "deposit", "field"};

struct pic_species {
    pic_sim *sim = nullptr;
    cudaStream_t stream = nullptr;     // where this species' kernels go: the sim's stream, or -- for the duration of a
                                       // pic_push_all -- its own (own_stream), so that the species' steps overlap
    cudaStream_t own_stream = nullptr;
    cudaEvent_t join_ev = nullptr;
    long long cyc_step0 = 0;           // pic_cycle: step count before the first cycle that is still unverified
    bool chain_valid = false;          // push_fused: the library's last kernel launch was this species' commit kernel
    unsigned long long chain_mark = 0; // ... when sim->launches still has this value
    PushConst k{};
    double qm = 0;
    long long n_ub = 0, capacity = 0; // host-known upper bound of DevState::n
    double *x[2]{}, *vx[2]{}, *vy[2]{}, *vz[2]{};
    int *cell[2]{};
    int cur = 0; // active buffer set
    int arrange_every = 0;
    DevState *d_st = nullptr;
    int *d_count[2]{}, *d_off[2]{};
    int cur_off = 0; // d_off[cur_off] / d_count[cur_off] describe the last arrange
    unsigned long long *d_scan = nullptr;
    size_t scan_words = 0;
    // fused push+arrange step (fused.cuh)
    double2 *d_cs = nullptr;           // deposition: per-cell partial sums (allocated at the first pic_deposit)
    int h_maxcount = 0;                // bound of the largest per-cell count last seen by the host (sizes the fused tiles)
    int h_maxdef = 0;                  // most right-movers of one cell deferred to the next tile, last seen (sizes their queue)
    // asynchronous telemetry of the fused path: every few fused steps the device state is copied to pinned host
    // memory without waiting; push_fused reads the latest copy that has landed (the largest per-cell count drifts
    // over a long pic_push without any synchronising call, and a cell that outgrows the tile declines the step)
    DevState *h_tel = nullptr;
    cudaEvent_t tel_ev = nullptr;
    bool tel_pending = false;
    long long tel_step = 0;            // fused steps since the last telemetry copy was enqueued
    int h_abort_reason = 0;
    bool fused_off = false;            // the device reported a declined fused step (sticky)
    // fused steps enqueued but not yet verified (verify_fused): how many, and the host state when the run began
    long long unv_steps = 0, unv_steps0 = 0;
    long long declined_at = 0;         // step count when the last decline was detected
    int unv_cur0 = 0, unv_off0 = 0;
    // host-side conservative bound on cell displacement since the last arrange (decides whether the
    // general-path kernels need to be enqueued at all)
    double vkick = 0;                  // 2*|h|*max|E| of the field in force now
    double h_vmax = 0;                 // speed bound at the last sync
    double h_kick_acc = 0;             // sum of the per-step kicks of the steps enqueued since the last sync (the field
                                       // may change between steps: each step is bounded with the field it ran under)
    long long h_steps_since_sync = 0;
    long long h_wsum = 0;              // sum of per-step displacement bounds since the last arrange
    bool h_grouped = false;
    void *ws = nullptr;
    size_t ws_bytes = 0;
    long long steps = 0, steps_at_last_flux = 0;
    unsigned long long wall_last[2]{};
    bool counts_fresh = false; // count/offset describe the current state
    bool all_live = true;      // no flagged-dead particle in [0, n)
    bool reset_w = false;      // an arrange ran since the displacement bound was last folded
    int trace_last[6] = {-1, -1, -1, -1, -1, -1}; // PIC_TRACE: the launch geometry last reported
};

struct pic_sim {
    cudaStream_t stream = nullptr;
    double *d_E = nullptr;
    int nc = 0, periodic = 0;
    double dx = 0, dt = 0;
    double B[3]{};
    double Emax = 0; // max |E_node|
    bool emax_known = true; // false after the field was replaced on the device until the next sync reads its max |E|
    // field solve (field.cuh): library-owned scratch, allocated at the first pic_solve_field / pic_set_field_device
    double *d_f[2]{}, *d_phi = nullptr, *d_tile = nullptr, *d_scal = nullptr;
    unsigned long long *d_emax = nullptr;
    int device = 0;
    cudaEvent_t fork_ev = nullptr; // pic_push_all: the species' own streams start behind it
    // pic_cycle: cycles enqueued without a host check (fused steps + deposition + field solve), to be verified -- and,
    // should a fused step have declined, redone from that cycle on -- by the next synchronising call
    struct CycleRec { int ncycles; std::vector<double> w; int passes; double *rho, *phi; };
    std::vector<CycleRec> cyc_pending;
    int *d_frozen = nullptr;       // device flag: a fused step of a pending cycle declined (fused.cuh, field.cuh)
    bool in_cycle = false;         // push_fused hands d_frozen to its kernels
    std::vector<pic_species *> sp;
    unsigned long long launches = 0;
    int opt_fused = 1, opt_timing = 0, opt_tile_scatter = 1, opt_fused_tma = 1, opt_fused_pdl = 1, opt_fused_taper = -1, opt_species_streams = 1, opt_cycle_async = 1, opt_field_fused = 1, opt_field_bps = 0;
    int field_grid_max = 0; // resident blocks of field_solve_kernel (cooperative launch)
    int opt_fused_cpc = 0, opt_fused_rows = 0, opt_fused_slots = 0, opt_fused_stages = 0; // tuning knobs of the fused step (0 = automatic)
    int sm_count = 148;
    // per-kernel device timing (option "kernel_timing"): event pairs recorded around launches
    struct Span { int id; cudaEvent_t a, b; };
    std::vector<Span> spans;
    std::vector<cudaEvent_t> free_events;
    double k_ms[K_COUNT] = {};
    unsigned long long k_launches[K_COUNT] = {};
};

// NVTX range for the lifetime of the object (ranges "mover", "hist", "scan", "scatter", ... per
// kernel class, plus one per multi-phase API call).
struct NvtxRange {
    explicit NvtxRange(const char *name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
    NvtxRange(const NvtxRange &) = delete;
    NvtxRange &operator=(const NvtxRange &) = delete;
};

// Records an event pair around the launches made during its lifetime (only when timing is on), inside an NVTX range
// named after the kernel class.
struct KernelSpan {
    pic_sim *sim;
    cudaEvent_t a = nullptr, b = nullptr;
    int id;
    static cudaEvent_t get(pic_sim *sim)
    {
        if (!sim->free_events.empty()) { cudaEvent_t e = sim->free_events.back(); sim->free_events.pop_back(); return e; }
        cudaEvent_t e = nullptr;
        if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); return nullptr; }
        return e;
    }
    cudaStream_t stream;
    KernelSpan(pic_sim *s, int kid, cudaStream_t st = nullptr) : sim(s), id(kid), stream(st ? st : s->stream)
    {
        nvtxRangePushA(K_NAMES[kid]);
        if (!sim->opt_timing) return;
        a = get(sim); b = get(sim);
        if (a) cudaEventRecord(a, stream);
    }
    ~KernelSpan()
    {
        nvtxRangePop();
        if (!a || !b) return;
        cudaEventRecord(b, stream);
        sim->spans.push_back({id, a, b});
    }
};

static bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// Device memory the library owns (handles' small objects, field scratch, the arena of pic_run_host) comes from one
// stream-ordered memory pool per device that keeps what is freed instead of returning it to the driver: PAPER.md:89
// "allocate once, keep resident, release at the end", applied across calls -- a second pic_create / pic_run_host of
// the same size costs no cudaMalloc and no cudaFree (both synchronise the device and take milliseconds for
// gigabytes).  pic_trim_memory() hands the cached memory back.
static cudaMemPool_t g_pool[64] = {};
static std::vector<void *> g_pinned_free; // pinned DevState blocks of destroyed species (telemetry), reused
// The arena of pic_run_host (gigabytes: two buffer sets and the workspace of every species) is a plain cudaMalloc
// kept for the next call -- growing a memory pool by 9 GB took 1.15 s against 1-2 ms for cudaMalloc.
static struct { char *p; size_t bytes; bool in_use; } g_arena[64] = {};

static std::mutex g_mem_mu; // guards g_pool / g_pinned_free / g_arena (sims of different threads share them)
static bool g_pool_broken[64] = {}; // the device or driver has no memory pools: plain cudaMalloc from then on

static cudaError_t dev_alloc(void **p, size_t bytes, int device, cudaStream_t st)
{
    *p = nullptr;
    cudaMemPool_t pool = nullptr;
    if (device >= 0 && device < 64) {
        std::lock_guard<std::mutex> lock(g_mem_mu);
        if (!g_pool[device] && !g_pool_broken[device]) {
            cudaMemPoolProps props{};
            props.allocType = cudaMemAllocationTypePinned;
            props.handleTypes = cudaMemHandleTypeNone;
            props.location.type = cudaMemLocationTypeDevice;
            props.location.id = device;
            unsigned long long keep = ~0ull;
            if (cudaMemPoolCreate(&g_pool[device], &props) != cudaSuccess ||
                cudaMemPoolSetAttribute(g_pool[device], cudaMemPoolAttrReleaseThreshold, &keep) != cudaSuccess) {
                cudaGetLastError();
                if (g_pool[device]) cudaMemPoolDestroy(g_pool[device]);
                g_pool[device] = nullptr;
                g_pool_broken[device] = true;
            }
        }
        pool = g_pool[device];
    }
    if (!pool) return cudaMalloc(p, bytes ? bytes : 16); // dev_free's cudaFreeAsync takes these too
    return cudaMallocFromPoolAsync(p, bytes ? bytes : 16, pool, st);
}

template <typename T>
static cudaError_t dev_alloc(T **p, size_t bytes, int device, cudaStream_t st)
{
    return dev_alloc(reinterpret_cast<void **>(p), bytes, device, st);
}

static void dev_free(void *p, cudaStream_t st)
{
    if (p) cudaFreeAsync(p, st);
}

extern "C" int pic_trim_memory(void)
{
    int dev = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceSynchronize());
    std::lock_guard<std::mutex> lock(g_mem_mu);
    if (dev >= 0 && dev < 64 && g_pool[dev]) CU(cudaMemPoolTrimTo(g_pool[dev], 0));
    if (dev >= 0 && dev < 64 && g_arena[dev].p && !g_arena[dev].in_use) {
        CU(cudaFree(g_arena[dev].p));
        g_arena[dev].p = nullptr;
        g_arena[dev].bytes = 0;
    }
    for (void *h : g_pinned_free) cudaFreeHost(h);
    g_pinned_free.clear();
    return PIC_OK;
}

extern "C" const char *pic_strerror(int s)
{
    switch (s) {
    case PIC_OK: return "ok";
    case PIC_EINVAL: return "invalid argument";
    case PIC_ENOMEM: return "out of memory";
    case PIC_ECUDA: return "CUDA error";
    case PIC_ECAPACITY: return "capacity or workspace too small";
    case PIC_ESTATE: return "invalid state";
    default: return "unknown status";
    }
}
extern "C" const char *pic_last_error(void) { return g_err; }

extern "C" size_t pic_workspace_bytes(int32_t nc, int64_t capacity)
{
    (void)nc;
    if (capacity < 0) return 0;
    return std::max(general_workspace_bytes((long long)capacity), ts_workspace_bytes((long long)capacity));
}

static void free_species(pic_species *s)
{
    if (!s) return;
    cudaStream_t st = s->sim ? s->sim->stream : nullptr;
    dev_free(s->d_st, st);
    for (int b = 0; b < 2; ++b) { dev_free(s->d_count[b], st); dev_free(s->d_off[b], st); }
    dev_free(s->d_scan, st);
    dev_free(s->d_cs, st);
    if (s->h_tel) {
        std::lock_guard<std::mutex> lock(g_mem_mu);
        g_pinned_free.push_back(s->h_tel);
    }
    if (s->tel_ev) cudaEventDestroy(s->tel_ev);
    if (s->join_ev) cudaEventDestroy(s->join_ev);
    if (s->own_stream) cudaStreamDestroy(s->own_stream);
    delete s;
}

extern "C" void pic_destroy(pic_sim *sim)
{
    if (!sim) return;
    cudaStreamSynchronize(sim->stream);
    for (pic_species *s : sim->sp) free_species(s);
    for (auto &sp : sim->spans) { cudaEventDestroy(sp.a); cudaEventDestroy(sp.b); }
    for (cudaEvent_t e : sim->free_events) cudaEventDestroy(e);
    if (sim->fork_ev) cudaEventDestroy(sim->fork_ev);
    dev_free(sim->d_E, sim->stream);
    dev_free(sim->d_f[0], sim->stream); dev_free(sim->d_f[1], sim->stream); dev_free(sim->d_phi, sim->stream);
    dev_free(sim->d_tile, sim->stream); dev_free(sim->d_scal, sim->stream);
    dev_free(sim->d_emax, sim->stream);
    dev_free(sim->d_frozen, sim->stream);
    cudaStreamSynchronize(sim->stream); // the frees are stream-ordered: the memory is back in the pool on return
    delete sim;
}

// Per-species Boris constants, DESIGN.md section 3 (each line one rounded operation; host
// code is compiled with -ffp-contract=off).
static void boris_constants(double qm, double dt, double dx, const double *B, PushConst &k)
{
    volatile double h = (qm * dt) * 0.5;
    volatile double tx = h * B[0], ty = h * B[1], tz = h * B[2];
    volatile double txx = tx * tx, tyy = ty * ty, tzz = tz * tz;
    volatile double t2a = txx + tyy;
    volatile double t2 = t2a + tzz;
    volatile double den = 1.0 + t2;
    volatile double f = 2.0 / den;
    k.h = h; k.tx = tx; k.ty = ty; k.tz = tz;
    volatile double sx = f * tx, sy = f * ty, sz = f * tz;
    k.sx = sx; k.sy = sy; k.sz = sz;
    volatile double inv = 1.0 / dx;
    k.inv_dx = inv;
    k.dt = dt;
}

static int launch_check(pic_sim *sim, const char *what)
{
    sim->launches++;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, what);
    return PIC_OK;
}

static int status_to_rc(int status)
{
    if (status & ERR_BAD_INITIAL) return PIC_ESTATE;
    if (status & ERR_OUT_OF_DOMAIN) return PIC_ESTATE;
    if (status & ERR_ARRANGE_SKIPPED) return PIC_ESTATE;
    if (status & ERR_NEED_WORKSPACE) return PIC_ECAPACITY;
    return PIC_OK;
}

static int run_scan(pic_species *s, const int *in, int *out, int m, ScanFold fold)
{
    pic_sim *sim = s->sim;
    size_t words = scan_scratch_words(m);
    CU(cudaMemsetAsync(s->d_scan, 0, words * sizeof(unsigned long long), s->stream));
    int ntiles = (m + SCAN_TILE - 1) / SCAN_TILE;
    KernelSpan span(sim, K_SCAN, s->stream);
    scan_exclusive_kernel<<<ntiles, SCAN_THREADS, 0, s->stream>>>(in, out, m, s->d_scan, fold);
    return launch_check(sim, "scan_exclusive_kernel");
}

static float bits_to_float(unsigned u)
{
    float f;
    memcpy(&f, &u, sizeof f);
    return f;
}

// raise DevState::maxcount to the largest per-cell count of the offsets in slot `which`
static int run_maxcount(pic_species *s, int which)
{
    pic_sim *sim = s->sim;
    const int nc = sim->nc;
    maxcount_kernel<<<(nc + 255) / 256, 256, 0, s->stream>>>(s->d_off[which], nc, s->d_st);
    return launch_check(sim, "maxcount_kernel");
}

static int fused_rows(const pic_species *s, int *ctas_per_sm);
static int verify_fused(pic_species *s);

static bool fused_possible(const pic_species *s)
{
    return s->sim->opt_fused && !s->fused_off && s->arrange_every == 1 && s->sim->nc >= FUSED_MIN_NC &&
           fused_rows(s, nullptr) > 0;
}

// Host-side bound (cells) on what one more mover step can displace any particle.
static long long host_step_bound(pic_species *s)
{
    if (!s->sim->emax_known) return 1LL << 40; // the field was replaced on the device: no bound until the next sync
    const double v = s->h_vmax * (1.0 + 1e-6) + s->h_kick_acc + s->vkick;
    const double reach = v * s->k.dt * s->k.inv_dx;
    if (!(reach < 1e9)) return 1LL << 40;
    return (long long)std::ceil(reach + 1e-9) + 1;
}

// The instance of fused_kernel for a launch geometry.
template <int R, int D>
static void (*fused_pick_rd(bool periodic, bool bz0, bool tma))(FusedArgs)
{
    if (D != FUSED_DEF) // the large queue exists for the TMA kernels only
        return periodic ? (bz0 ? fused_kernel<R, true, true, true, D> : fused_kernel<R, true, false, true, D>)
                        : (bz0 ? fused_kernel<R, false, true, true, D> : fused_kernel<R, false, false, true, D>);
    return periodic ? (bz0 ? (tma ? fused_kernel<R, true, true, true, FUSED_DEF> : fused_kernel<R, true, true, false, FUSED_DEF>)
                           : (tma ? fused_kernel<R, true, false, true, FUSED_DEF> : fused_kernel<R, true, false, false, FUSED_DEF>))
                    : (bz0 ? (tma ? fused_kernel<R, false, true, true, FUSED_DEF> : fused_kernel<R, false, true, false, FUSED_DEF>)
                           : (tma ? fused_kernel<R, false, false, true, FUSED_DEF> : fused_kernel<R, false, false, false, FUSED_DEF>));
}

static void (*fused_pick(int rows, bool periodic, bool bz0, bool tma, int def))(FusedArgs)
{
    if (def != FUSED_DEF)
        return rows == 8 ? fused_pick_rd<8, FUSED_DEF_BIG>(periodic, bz0, tma)
             : rows == 12 ? fused_pick_rd<12, FUSED_DEF_BIG>(periodic, bz0, tma) : fused_pick_rd<16, FUSED_DEF_BIG>(periodic, bz0, tma);
    return rows == 8 ? fused_pick_rd<8, FUSED_DEF>(periodic, bz0, tma)
         : rows == 12 ? fused_pick_rd<12, FUSED_DEF>(periodic, bz0, tma) : fused_pick_rd<16, FUSED_DEF>(periodic, bz0, tma);
}

// The fused kernels need more dynamic shared memory than the default limit: raise it once per DEVICE (the attribute
// is per device and per function; a process may create sims on several devices).
static std::mutex g_attr_mu;
static int fused_set_attributes(int device)
{
    static bool done[64] = {};
    std::lock_guard<std::mutex> lock(g_attr_mu); // sims of different threads may be created at the same time
    if (device >= 0 && device < 64 && done[device]) return PIC_OK;
    std::vector<void (*)(FusedArgs)> kerns;
    for (int rows : {8, 12, 16})
        for (int per = 0; per < 2; ++per)
            for (int bz0 = 0; bz0 < 2; ++bz0)
                for (int tma = 0; tma < 2; ++tma)
                    for (int def : {FUSED_DEF, FUSED_DEF_BIG})
                        if (tma || def == FUSED_DEF) kerns.push_back(fused_pick(rows, per != 0, bz0 != 0, tma != 0, def));
    for (auto kfn : kerns) CU(cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
    CU(cudaFuncSetAttribute(tile_scatter_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TS_SMEM_BYTES));
    if (device >= 0 && device < 64) done[device] = true;
    return PIC_OK;
}

// ------------------------------------------------------------------------------------------
// create
// ------------------------------------------------------------------------------------------
// Host-side half of creating a species: argument checks and every allocation, no wait on the stream (so that it
// overlaps whatever the caller has in flight on it, e.g. the uploads of pic_run_host).
static int alloc_species(pic_sim *sim, const pic_species_desc &d, pic_species **out)
{
    if (!std::isfinite(d.qm) || d.n < 0 || d.capacity < 0 || d.arrange_every < 0) return PIC_EINVAL;
    if (d.n > d.capacity) return PIC_ECAPACITY;
    if (d.capacity >= (1LL << 31) - 64) return PIC_ECAPACITY;
    for (int b = 0; b < 2; ++b) {
        if (d.capacity > 0 && (!d.x[b] || !d.vx[b] || !d.vy[b] || !d.vz[b] || !d.cell[b])) return PIC_EINVAL;
        if (!aligned16(d.x[b]) || !aligned16(d.vx[b]) || !aligned16(d.vy[b]) || !aligned16(d.vz[b]) ||
            !aligned16(d.cell[b]))
            return PIC_EINVAL;
    }
    if ((d.workspace == nullptr) != (d.workspace_bytes == 0)) return PIC_EINVAL;
    if (d.workspace && (reinterpret_cast<uintptr_t>(d.workspace) & 255u)) return PIC_EINVAL;

    pic_species *s = new (std::nothrow) pic_species;
    if (!s) return PIC_ENOMEM;
    *out = s;
    s->sim = sim;
    s->stream = sim->stream;
    s->qm = d.qm;
    s->n_ub = d.n;
    s->capacity = d.capacity;
    for (int b = 0; b < 2; ++b) {
        s->x[b] = d.x[b]; s->vx[b] = d.vx[b]; s->vy[b] = d.vy[b]; s->vz[b] = d.vz[b]; s->cell[b] = d.cell[b];
    }
    s->arrange_every = d.arrange_every;
    s->ws = d.workspace;
    s->ws_bytes = d.workspace_bytes;
    boris_constants(d.qm, sim->dt, sim->dx, sim->B, s->k);
    s->k.nc = sim->nc;
    s->k.periodic = sim->periodic;
    s->k.L = (double)sim->nc * sim->dx;

    const int nc = sim->nc;
    CU(dev_alloc(&s->d_st, sizeof(DevState), sim->device, sim->stream));
    for (int b = 0; b < 2; ++b) {
        CU(dev_alloc(&s->d_count[b], sizeof(int) * ((size_t)nc + 16), sim->device, sim->stream));
        CU(dev_alloc(&s->d_off[b], sizeof(int) * ((size_t)nc + 16), sim->device, sim->stream));
        CU(cudaMemsetAsync(s->d_count[b], 0, sizeof(int) * ((size_t)nc + 16), sim->stream));
        CU(cudaMemsetAsync(s->d_off[b], 0, sizeof(int) * ((size_t)nc + 16), sim->stream));
    }
    // scan scratch sized for the largest array the library scans (per-cell counts, or the
    // general path's per-tile digit histograms)
    long long max_scan = std::max<long long>((long long)nc + 1, general_scan_elems(d.capacity));
    s->scan_words = scan_scratch_words(max_scan);
    CU(dev_alloc(&s->d_scan, s->scan_words * sizeof(unsigned long long), sim->device, sim->stream));
    {
        std::lock_guard<std::mutex> lock(g_mem_mu);
        if (!g_pinned_free.empty()) { s->h_tel = static_cast<DevState *>(g_pinned_free.back()); g_pinned_free.pop_back(); }
    }
    if (!s->h_tel) CU(cudaMallocHost(&s->h_tel, sizeof(DevState)));
    CU(cudaEventCreateWithFlags(&s->tel_ev, cudaEventDisableTiming));
    return PIC_OK;
}

// Stream-side half: validate the initial state on the device, build its per-cell count / offset.  Syncs.
static int init_species(pic_sim *sim, pic_species *s, const pic_species_desc &d)
{
    const int nc = sim->nc;
    DevState h{};
    h.n = (int)d.n;
    CU(cudaMemcpyAsync(s->d_st, &h, sizeof h, cudaMemcpyHostToDevice, s->stream));
    CU(cudaStreamSynchronize(s->stream)); // h is a stack object

    // validate the initial state, build count/offset of the initial grouping
    if (d.n > 0) {
        int blocks = (int)((d.n + 255) / 256);
        validate_kernel<<<blocks, 256, 0, s->stream>>>(s->x[0], s->vx[0], s->vy[0], s->vz[0], s->cell[0], s->k, s->d_st);
        if (int rc = launch_check(sim, "validate_kernel")) return rc;
    }
    CU(cudaMemcpyAsync(&h, s->d_st, sizeof h, cudaMemcpyDeviceToHost, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    if (h.status & ERR_BAD_INITIAL) {
        snprintf(g_err, sizeof g_err, "initial state violates 0<=x<L, cell==floor(x/dx), all live");
        return PIC_ESTATE;
    }
    bool grouped = !(h.status & ERR_NOT_GROUPED);
    if (d.n > 0) {
        int blocks = (int)((d.n + HIST_THREADS * HIST_ITEMS - 1) / (HIST_THREADS * HIST_ITEMS));
        hist_kernel<<<blocks, HIST_THREADS, 0, s->stream>>>(s->cell[0], s->d_count[0], s->d_st);
        if (int rc = launch_check(sim, "hist_kernel")) return rc;
    }
    ScanFold nofold{nullptr, 0, 0, 0, nullptr};
    if (int rc = run_scan(s, s->d_count[0], s->d_off[0], nc, nofold)) return rc;
    s->vkick = 2.0 * std::fabs(s->k.h) * sim->Emax;
    s->h_vmax = std::sqrt((double)bits_to_float(h.vmax2));
    s->h_grouped = grouped;
    h.status = 0;
    h.w_acc = grouped ? 0 : W_UNKNOWN;
    CU(cudaMemcpyAsync(s->d_st, &h, sizeof h, cudaMemcpyHostToDevice, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    if (grouped) { // largest per-cell count: sizes the tiles of the fused step
        if (int rc = run_maxcount(s, 0)) return rc;
        CU(cudaMemcpyAsync(&h, s->d_st, sizeof h, cudaMemcpyDeviceToHost, s->stream));
        CU(cudaStreamSynchronize(s->stream));
        s->h_maxcount = h.maxcount;
    }
    s->cur = 0;
    s->cur_off = 0;
    s->counts_fresh = grouped;
    s->all_live = true;
    s->reset_w = false;
    if (int rc = fused_set_attributes(sim->device)) return rc;
    return PIC_OK;
}

extern "C" int pic_create(const pic_grid_desc *g, const pic_species_desc *species, int nspecies, pic_sim **out)
{
    if (out) *out = nullptr;
    if (!g || !species || !out || nspecies < 1) return PIC_EINVAL;
    if (g->nc < 1 || g->nc >= (1 << 30) || !g->E_nodes) return PIC_EINVAL;
    if (!(g->dx > 0) || !(g->dt > 0) || !std::isfinite(g->dx) || !std::isfinite(g->dt)) return PIC_EINVAL;
    if (g->boundary != PIC_PERIODIC && g->boundary != PIC_ABSORBING) return PIC_EINVAL;
    for (int a = 0; a < 3; ++a)
        if (!std::isfinite(g->B[a])) return PIC_EINVAL;
    double emax = 0;
    for (int j = 0; j <= g->nc; ++j) {
        if (!std::isfinite(g->E_nodes[j])) return PIC_EINVAL;
        emax = std::max(emax, std::fabs(g->E_nodes[j]));
    }

    int dev = 0;
    CU(cudaGetDevice(&dev));
    pic_sim *sim = new (std::nothrow) pic_sim;
    if (!sim) return PIC_ENOMEM;
    sim->stream = static_cast<cudaStream_t>(g->stream);
    sim->device = dev;
    sim->nc = g->nc;
    sim->periodic = g->boundary == PIC_PERIODIC;
    sim->dx = g->dx;
    sim->dt = g->dt;
    for (int a = 0; a < 3; ++a) sim->B[a] = g->B[a];
    sim->Emax = emax;
    int rc = PIC_OK;
    do {
        cudaError_t e = cudaDeviceGetAttribute(&sim->sm_count, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) { rc = cuda_fail(e, "cudaDeviceGetAttribute"); break; }
        // E padded to an even number of nodes (+2) so that 16-byte bulk copies of any window stay inside
        e = dev_alloc(&sim->d_E, sizeof(double) * ((size_t)g->nc + 8), sim->device, sim->stream);
        if (e != cudaSuccess) { rc = e == cudaErrorMemoryAllocation ? PIC_ENOMEM : cuda_fail(e, "cudaMalloc E"); break; }
        for (int i = 0; i < nspecies && rc == PIC_OK; ++i) { // all allocations first: nothing here waits on the stream
            pic_species *s = nullptr;
            rc = alloc_species(sim, species[i], &s);
            if (s) sim->sp.push_back(s);
        }
        if (rc != PIC_OK) break;
        e = cudaMemsetAsync(sim->d_E, 0, sizeof(double) * ((size_t)g->nc + 8), sim->stream);
        if (e != cudaSuccess) { rc = cuda_fail(e, "cudaMemsetAsync E"); break; }
        e = cudaMemcpyAsync(sim->d_E, g->E_nodes, sizeof(double) * ((size_t)g->nc + 1), cudaMemcpyHostToDevice, sim->stream);
        if (e != cudaSuccess) { rc = cuda_fail(e, "cudaMemcpyAsync E"); break; }
        e = cudaStreamSynchronize(sim->stream);
        if (e != cudaSuccess) { rc = cuda_fail(e, "cudaStreamSynchronize"); break; }
        for (int i = 0; i < nspecies && rc == PIC_OK; ++i) rc = init_species(sim, sim->sp[i], species[i]);
    } while (0);
    if (rc != PIC_OK) {
        pic_destroy(sim);
        return rc;
    }
    *out = sim;
    return PIC_OK;
}

extern "C" pic_species *pic_species_at(pic_sim *sim, int i)
{
    if (!sim || i < 0 || i >= (int)sim->sp.size()) return nullptr;
    return sim->sp[i];
}

static int verify_cycles(pic_sim *sim);

extern "C" int pic_set_field(pic_sim *sim, const double *E)
{
    if (!sim || !E) return PIC_EINVAL;
    for (pic_species *s : sim->sp) // steps already enqueued must have run (or be redone) with the old field
        if (int rc = verify_fused(s)) return rc;
    double emax = 0;
    for (int j = 0; j <= sim->nc; ++j) {
        if (!std::isfinite(E[j])) return PIC_EINVAL;
        emax = std::max(emax, std::fabs(E[j]));
    }
    sim->Emax = emax;
    sim->emax_known = true;
    for (pic_species *s : sim->sp) s->vkick = 2.0 * std::fabs(s->k.h) * emax;
    CU(cudaMemcpyAsync(sim->d_E, E, sizeof(double) * ((size_t)sim->nc + 1), cudaMemcpyHostToDevice, sim->stream));
    CU(cudaStreamSynchronize(sim->stream)); // E is a caller buffer that may be pageable
    return PIC_OK;
}

// scratch of the field solve, allocated on first use
static int field_alloc(pic_sim *sim)
{
    if (sim->d_emax) return PIC_OK;
    const size_t nb = sizeof(double) * ((size_t)sim->nc + 8);
    const size_t nt = (size_t)fld_ntiles(sim->nc);
    cudaError_t e = dev_alloc(&sim->d_f[0], nb, sim->device, sim->stream);
    if (e == cudaSuccess) e = dev_alloc(&sim->d_f[1], nb, sim->device, sim->stream);
    if (e == cudaSuccess) e = dev_alloc(&sim->d_phi, nb, sim->device, sim->stream);
    if (e == cudaSuccess) e = dev_alloc(&sim->d_tile, sizeof(double) * 4 * nt, sim->device, sim->stream);
    if (e == cudaSuccess) e = dev_alloc(&sim->d_scal, sizeof(double) * 4, sim->device, sim->stream);
    if (e == cudaSuccess) e = dev_alloc(&sim->d_emax, 2 * sizeof(unsigned long long), sim->device, sim->stream); // max |E| bits, two tickets
    if (e == cudaSuccess) e = cudaMemsetAsync(sim->d_emax, 0, 2 * sizeof(unsigned long long), sim->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(sim->d_scal, 0, sizeof(double) * 4, sim->stream);
    if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? PIC_ENOMEM : cuda_fail(e, "cudaMalloc field scratch");
    return PIC_OK;
}

// steps already enqueued must have run (or be redone by the split kernels) with the field they were issued under
static int field_barrier(pic_sim *sim)
{
    for (pic_species *s : sim->sp)
        if (int rc = verify_fused(s)) return rc;
    return PIC_OK;
}

extern "C" int pic_set_field_device(pic_sim *sim, const double *E_dev)
{
    if (!sim || !E_dev) return PIC_EINVAL;
    if (int rc = field_barrier(sim)) return rc;
    if (int rc = field_alloc(sim)) return rc;
    const int nc = sim->nc;
    CU(cudaMemcpyAsync(sim->d_E, E_dev, sizeof(double) * ((size_t)nc + 1), cudaMemcpyDeviceToDevice, sim->stream));
    CU(cudaMemsetAsync(sim->d_emax, 0, sizeof(unsigned long long), sim->stream));
    KernelSpan span(sim, K_FIELD);
    field_emax_kernel<<<(nc + 1 + FLD_THREADS - 1) / FLD_THREADS, FLD_THREADS, 0, sim->stream>>>(sim->d_E, nc, sim->d_emax);
    if (int rc = launch_check(sim, "field_emax_kernel")) return rc;
    sim->emax_known = false;
    return PIC_OK;
}

static int solve_enqueue(pic_sim *sim, const double *rho_dev, int smooth_passes, double *phi_dev, const int *frozen);

extern "C" int pic_solve_field(pic_sim *sim, const double *rho_dev, int smooth_passes, double *phi_dev)
{
    if (!sim || !rho_dev || smooth_passes < 0 || smooth_passes > 1024) return PIC_EINVAL;
    if (sim->nc < 2) return PIC_EINVAL;
    if (int rc = field_barrier(sim)) return rc;
    return solve_enqueue(sim, rho_dev, smooth_passes, phi_dev, nullptr);
}

// The kernels of one field solve, enqueued on the sim's stream without any host-side check.
static int solve_enqueue(pic_sim *sim, const double *rho_dev, int smooth_passes, double *phi_dev, const int *frozen)
{
    if (int rc = field_alloc(sim)) return rc;
    const int nc = sim->nc;
    const int nblk = (nc + 1 + FLD_THREADS - 1) / FLD_THREADS;
    KernelSpan span(sim, K_FIELD);
    FieldArgs a{};
    a.phi = sim->d_phi; a.E = sim->d_E; a.phi_out = phi_dev;
    a.ntiles = fld_ntiles(nc);
    a.tile_s = sim->d_tile; a.tile_t = sim->d_tile + a.ntiles; a.tile_sum = sim->d_tile + 2 * (size_t)a.ntiles;
    a.tile_lo = sim->d_tile + 3 * (size_t)a.ntiles;
    a.scal = sim->d_scal; a.emax_bits = sim->d_emax;
    a.ticket = reinterpret_cast<unsigned *>(sim->d_emax + 1);
    a.nc = nc; a.periodic = sim->periodic;
    a.frozen = frozen;
    { volatile double d2 = sim->dx * sim->dx; a.dx2 = d2; volatile double inv = 1.0 / sim->dx; a.inv_dx = inv; }
    if (sim->opt_field_fused) {
        // one cooperative kernel: a grid of resident blocks walks the phases and meets at grid-wide barriers
        if (sim->field_grid_max == 0) {
            int per_sm = 0;
            CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, field_solve_kernel, FLD_THREADS, 0));
            sim->field_grid_max = std::max(1, per_sm * sim->sm_count);
        }
        // blocks per SM: the barrier costs more with more blocks, the phases less
        const int want = sim->opt_field_bps ? sim->opt_field_bps : (nc > 400000 ? 4 : 1);
        int grid = std::max(1, std::min(std::min(sim->field_grid_max, want * sim->sm_count), nblk));
        const double *rho_in = rho_dev;
        double *f0 = sim->d_f[0], *f1 = sim->d_f[1];
        int passes = smooth_passes;
        void *args[] = {&a, &rho_in, &f0, &f1, &passes};
        CU(cudaLaunchCooperativeKernel((const void *)field_solve_kernel, dim3((unsigned)grid), dim3(FLD_THREADS), args, 0, sim->stream));
        if (int rc = launch_check(sim, "field_solve_kernel")) return rc;
        sim->emax_known = false;
        return PIC_OK;
    }
    const double *rho = rho_dev;
    for (int p = 0; p < smooth_passes; ++p) {
        double *out = sim->d_f[p & 1];
        field_smooth_kernel<<<nblk, FLD_THREADS, 0, sim->stream>>>(rho, out, nc, sim->periodic);
        if (int rc = launch_check(sim, "field_smooth_kernel")) return rc;
        rho = out;
    }
    a.rho = rho;
    CU(cudaMemsetAsync(sim->d_emax, 0, sizeof(unsigned long long), sim->stream));
    if (sim->periodic) {
        field_sum_kernel<<<a.ntiles, FLD_THREADS, 0, sim->stream>>>(a);
        if (int rc = launch_check(sim, "field_sum_kernel")) return rc;
    }
    field_tile_kernel<<<a.ntiles, FLD_THREADS, 0, sim->stream>>>(a);
    if (int rc = launch_check(sim, "field_tile_kernel")) return rc;
    field_chain_kernel<<<1, FLD_THREADS, 0, sim->stream>>>(a);
    if (int rc = launch_check(sim, "field_chain_kernel")) return rc;
    field_phi_kernel<<<a.ntiles, FLD_THREADS, 0, sim->stream>>>(a);
    if (int rc = launch_check(sim, "field_phi_kernel")) return rc;
    field_e_kernel<<<nblk, FLD_THREADS, 0, sim->stream>>>(a);
    if (int rc = launch_check(sim, "field_e_kernel")) return rc;
    sim->emax_known = false;
    return PIC_OK;
}

extern "C" int pic_get_field(pic_sim *sim, double *E_host)
{
    if (!sim || !E_host) return PIC_EINVAL;
    if (!sim->cyc_pending.empty()) // unchecked pic_cycle work decides what the field is
        if (int rc = verify_cycles(sim)) return rc;
    CU(cudaMemcpyAsync(E_host, sim->d_E, sizeof(double) * ((size_t)sim->nc + 1), cudaMemcpyDeviceToHost, sim->stream));
    CU(cudaStreamSynchronize(sim->stream));
    return PIC_OK;
}

extern "C" int pic_set_option(pic_sim *sim, const char *key, int value)
{
    if (!sim || !key) return PIC_EINVAL;
    const bool flag = value == 0 || value == 1;
    if (!strcmp(key, "tile_scatter") && flag) sim->opt_tile_scatter = value;
    else if (!strcmp(key, "kernel_timing") && flag) sim->opt_timing = value;
    else if (!strcmp(key, "fused") && flag) sim->opt_fused = value;
    else if (!strcmp(key, "fused_tma") && flag) sim->opt_fused_tma = value;
    else if (!strcmp(key, "fused_pdl") && flag) sim->opt_fused_pdl = value;
    else if (!strcmp(key, "species_streams") && flag) sim->opt_species_streams = value;
    else if (!strcmp(key, "cycle_async") && flag) sim->opt_cycle_async = value;
    else if (!strcmp(key, "field_fused") && flag) sim->opt_field_fused = value;
    else if (!strcmp(key, "field_blocks_per_sm") && value >= 0 && value <= 8) sim->opt_field_bps = value;
    else if (!strcmp(key, "fused_taper") && value >= -1 && value < FUSED_SEGS) sim->opt_fused_taper = value;
    else if (!strcmp(key, "fused_cells_per_cta") && value >= 0 && value <= FUSED_CPC_MAX) sim->opt_fused_cpc = value;
    else if (!strcmp(key, "fused_stage_slots") && value >= 0 && value <= 512 && value % 2 == 0) sim->opt_fused_slots = value;
    else if (!strcmp(key, "fused_stages") && value >= 0 && value <= 2) sim->opt_fused_stages = value;
    else if (!strcmp(key, "fused_rows") && (value == 0 || value == 8 || value == 12 || value == 16)) sim->opt_fused_rows = value;
    else return PIC_EINVAL;
    return PIC_OK;
}

extern "C" int pic_kernel_time(pic_sim *sim, const char *kernel, double *ms_total, uint64_t *spans)
{
    if (!sim || !kernel) return PIC_EINVAL;
    int id = -1;
    for (int k = 0; k < K_COUNT; ++k)
        if (!strcmp(kernel, K_NAMES[k])) id = k;
    if (id < 0) return PIC_EINVAL;
    CU(cudaStreamSynchronize(sim->stream));
    for (auto &sp : sim->spans) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, sp.a, sp.b) == cudaSuccess) {
            sim->k_ms[sp.id] += ms;
            sim->k_launches[sp.id]++;
        } else {
            cudaGetLastError();
        }
        sim->free_events.push_back(sp.a);
        sim->free_events.push_back(sp.b);
    }
    sim->spans.clear();
    if (ms_total) *ms_total = sim->k_ms[id];
    if (spans) *spans = sim->k_launches[id];
    sim->k_ms[id] = 0;
    sim->k_launches[id] = 0;
    return PIC_OK;
}

extern "C" int pic_launch_count(pic_sim *sim, uint64_t *launches)
{
    if (!sim || !launches) return PIC_EINVAL;
    *launches = sim->launches;
    return PIC_OK;
}

// ------------------------------------------------------------------------------------------
// arrange (split path): [histogram] -> scan -> destination-driven scatter [-> general path]
// ------------------------------------------------------------------------------------------
// after_mover: a mover step ran since the last fold, so the scan's fold also commits its speed bound.
static int arrange_split(pic_species *s, bool hist_ready, bool after_mover)
{
    pic_sim *sim = s->sim;
    const int nc = sim->nc;
    const int src = s->cur, dst = s->cur ^ 1;
    const int oo = s->cur_off, on = s->cur_off ^ 1;
    if (!hist_ready) {
        CU(cudaMemsetAsync(s->d_count[on], 0, sizeof(int) * (size_t)nc, s->stream));
        if (s->n_ub > 0) {
            int blocks = (int)((s->n_ub + HIST_THREADS * HIST_ITEMS - 1) / (HIST_THREADS * HIST_ITEMS));
            KernelSpan span(sim, K_HIST, s->stream);
            hist_kernel<<<blocks, HIST_THREADS, 0, s->stream>>>(s->cell[src], s->d_count[on], s->d_st);
            if (int rc = launch_check(sim, "hist_kernel")) return rc;
        }
    }
    ScanFold fold{s->d_st, s->reset_w ? 1 : 0, 1, after_mover ? 1 : 0, nullptr};
    if (int rc = run_scan(s, s->d_count[on], s->d_off[on], nc, fold)) return rc;

    ScatterArgs a{};
    a.sx = s->x[src]; a.svx = s->vx[src]; a.svy = s->vy[src]; a.svz = s->vz[src]; a.scell = s->cell[src];
    a.dx = s->x[dst]; a.dvx = s->vx[dst]; a.dvy = s->vy[dst]; a.dvz = s->vz[dst]; a.dcell = s->cell[dst];
    a.off_old = s->d_off[oo]; a.count_new = s->d_count[on]; a.off_new = s->d_off[on];
    a.st = s->d_st; a.nc = nc; a.periodic = sim->periodic;
    a.w_limit = FAST_W_LIMIT;
    // general path: enqueued only if the host-side displacement bound cannot rule it out
    const bool general_follows = !(s->h_grouped && s->h_wsum <= FAST_W_LIMIT);
    a.general_follows = general_follows ? 1 : 0;
    {
        KernelSpan span(sim, K_SCATTER, s->stream);
        // tile-ranked stable scatter (tilesort.cuh) when the caller gave a workspace; the destination-driven
        // scatter behind it runs only if a tile declined (or instead of it without a workspace)
        const bool tiles = sim->opt_tile_scatter && s->ws && s->ws_bytes >= ts_workspace_bytes(s->n_ub) && s->n_ub > 0;
        if (tiles) {
            TileArgs t{};
            t.sx = a.sx; t.svx = a.svx; t.svy = a.svy; t.svz = a.svz; t.scell = a.scell;
            t.dx = a.dx; t.dvx = a.dvx; t.dvy = a.dvy; t.dvz = a.dvz; t.dcell = a.dcell;
            t.off_old = a.off_old; t.off_new = a.off_new; t.st = s->d_st;
            t.nc = nc; t.periodic = sim->periodic; t.w_limit = FAST_W_LIMIT;
            t.general_follows = a.general_follows;
            const int nt = (int)ts_ntiles(s->n_ub);
            t.tinfo = reinterpret_cast<int2 *>(s->ws);
            t.thist = reinterpret_cast<int *>(static_cast<char *>(s->ws) + (((size_t)(nt + 1) * sizeof(int2) + 255) & ~(size_t)255));
            tile_hist_kernel<<<nt, TS_THREADS, 0, s->stream>>>(t);
            if (int rc = launch_check(sim, "tile_hist_kernel")) return rc;
            tile_base_kernel<<<(nc + 255) / 256, 256, 0, s->stream>>>(t);
            if (int rc = launch_check(sim, "tile_base_kernel")) return rc;
            tile_scatter_kernel<<<nt, TS_THREADS, TS_SMEM_BYTES, s->stream>>>(t);
            if (int rc = launch_check(sim, "tile_scatter_kernel")) return rc;
            a.only_if = &s->d_st->tile_declined;
        }
        long long want = ((long long)nc + SCATTER_THREADS / 32 - 1) / (SCATTER_THREADS / 32);
        int blocks = (int)std::min<long long>(want, (long long)sim->sm_count * 64);
        scatter_fast_kernel<<<blocks, SCATTER_THREADS, 0, s->stream>>>(a);
        if (int rc = launch_check(sim, "scatter_fast_kernel")) return rc;
    }
    // every kernel of the general path returns at once unless scatter_fast_kernel declined on the device; if it is not
    // enqueued and the device declines after all (the host bound was wrong), ERR_ARRANGE_SKIPPED is raised
    if (general_follows) {
        GeneralArgs ga{};
        ga.sx = a.sx; ga.svx = a.svx; ga.svy = a.svy; ga.svz = a.svz; ga.scell = a.scell;
        ga.dx = a.dx; ga.dvx = a.dvx; ga.dvy = a.dvy; ga.dvz = a.dvz; ga.dcell = a.dcell;
        ga.st = s->d_st; ga.nc = nc; ga.n_ub = s->n_ub; ga.ws = s->ws; ga.ws_bytes = s->ws_bytes;
        ga.off_old = s->d_off[oo];
        ga.scan_scratch = s->d_scan;
        KernelSpan gspan(sim, K_GENERAL, s->stream); // general_arrange launches on the species' stream
        if (int rc = general_arrange(ga, s->stream, sim->sm_count, &sim->launches)) return rc == PIC_ECUDA ? cuda_fail(cudaGetLastError(), "general_arrange") : rc;
    }
    if (s->sim->opt_fused && s->arrange_every == 1)
        if (int rc = run_maxcount(s, on)) return rc;

    s->cur = dst;
    s->cur_off = on;
    s->counts_fresh = true;
    s->all_live = true;
    s->reset_w = true;
    s->h_wsum = 0;
    s->h_grouped = true;
    return PIC_OK;
}

extern "C" int pic_arrange(pic_species *s)
{
    if (!s) return PIC_EINVAL;
    if (int rc = verify_fused(s)) return rc;
    return arrange_split(s, false, false);
}

// ------------------------------------------------------------------------------------------
// push
// ------------------------------------------------------------------------------------------
template <bool RC, bool H>
static void launch_mover(pic_species *s, const MoverArgs &a, int blocks)
{
    mover_kernel<RC, H><<<blocks, MOVER_THREADS, 0, s->stream>>>(a);
}

static int push_split(pic_species *s, bool will_arrange)
{
    pic_sim *sim = s->sim;
    const int nc = sim->nc;
    const int on = s->cur_off ^ 1;
    if (will_arrange) CU(cudaMemsetAsync(s->d_count[on], 0, sizeof(int) * (size_t)nc, s->stream));
    if (s->n_ub > 0) {
        MoverArgs a{};
        a.x = s->x[s->cur]; a.vx = s->vx[s->cur]; a.vy = s->vy[s->cur]; a.vz = s->vz[s->cur];
        a.cell = s->cell[s->cur];
        a.E = sim->d_E; a.count = s->d_count[on]; a.st = s->d_st; a.k = s->k;
        long long pairs = (s->n_ub + 1) / 2;
        int blocks = (int)((pairs + MOVER_THREADS - 1) / MOVER_THREADS);
        const bool rc = !s->all_live;
        KernelSpan span(sim, K_MOVER, s->stream);
        if (rc) { if (will_arrange) launch_mover<true, true>(s, a, blocks); else launch_mover<true, false>(s, a, blocks); }
        else    { if (will_arrange) launch_mover<false, true>(s, a, blocks); else launch_mover<false, false>(s, a, blocks); }
        if (int r = launch_check(sim, "mover_kernel")) return r;
    }
    s->h_wsum = std::min<long long>(s->h_wsum + host_step_bound(s), 1LL << 40);
    s->h_steps_since_sync++;
    // a step enqueued while max |E| of a device-side field is still unknown has no known kick: the bound stays
    // "unknown" (infinite) until the next read_state refreshes the speed bound, even if pic_set_field intervenes
    s->h_kick_acc += s->sim->emax_known ? s->vkick : (double)INFINITY;
    if (!sim->periodic) s->all_live = false;
    s->counts_fresh = false;
    if (!will_arrange) {
        end_step_kernel<<<1, 1, 0, s->stream>>>(s->d_st, s->reset_w ? 1 : 0);
        s->reset_w = false;
        if (int r = launch_check(sim, "end_step_kernel")) return r;
    }
    return PIC_OK;
}

struct FusedGeom { int rows, slots, stages, cpc, ctas_per_sm, def, taper; size_t smem; };

// CTAs of fused_kernel<rows> an SM holds: registers (launch bounds of the instance) or shared memory.
static int fused_ctas_per_sm(int rows, int cpc, int stages, int def)
{
    const int by_regs = rows == 8 ? 16 : rows == 12 ? 12 : 8;
    const int by_smem = FUSED_SMEM_SM / (fused_layout(rows * 32, cpc, stages, def).total + 1024);
    return std::max(1, std::min(32, std::min(by_regs, by_smem)));
}

// Cells per CTA.  Every chunk pushes two halo cells on top of its own, and the grid runs in waves of
// sm_count * ctas_per_sm CTAs: pick the chunk size that wastes least to halo work and a ragged last wave.
static int fused_cells_per_cta(const pic_species *s, int rows, int stages, int def, int *taper)
{
    const pic_sim *sim = s->sim;
    *taper = std::max(sim->opt_fused_taper, 0);
    if (sim->opt_fused_cpc > 0) return sim->opt_fused_cpc;
    int best = FUSED_CPC_DEFAULT;
    {   // many waves: large chunks (little halo work), the last waves tapered (fused_schedule)
        const double resident = (double)sim->sm_count * fused_ctas_per_sm(rows, best, stages, def);
        if ((double)((sim->nc + best - 1) / best) >= 4.0 * resident) {
            if (sim->opt_fused_taper < 0) { *taper = FUSED_SEGS - 1; return FUSED_CPC_TAPER; }
            return best;
        }
    }
    // Species that step concurrently (inside pic_push_all each runs on a stream of its own) share the machine's CTA
    // slots: the waves are then counted over the chunks of ALL of them, a few waves beat two full ones (the species'
    // ramps and tails overlap), and a last wave with a little slack beats a packed one.  Measured at config 3
    // (profiles/r03_variants.md: 57 cells, the single-species optimum, 0.5435 ms; 39 / 23 cells 0.5162 / 0.5166 ms).
    const int conc = (s->own_stream && s->stream == s->own_stream) ? (int)sim->sp.size() : 1;
    double best_score = -1.0;
    for (int cpc = 2; cpc <= FUSED_CPC_SEARCH; ++cpc) {
        const double resident = (double)sim->sm_count * fused_ctas_per_sm(rows, cpc, stages, def);
        const double chunks = (double)((sim->nc + cpc - 1) / cpc);
        double score;
        if (conc == 1) {
            score = chunks / (std::ceil(chunks / resident) * resident) * cpc / (cpc + 2.0);
        } else {
            const double total = chunks * conc, waves = std::ceil(total / resident);
            double fill = total / (waves * resident);
            if (fill > 0.97) fill = 0.97 - 0.5 * (fill - 0.97);
            score = fill * cpc / (cpc + 2.0) * waves / (waves + 0.35);
        }
        if (score > best_score * 1.0001) { best_score = score; best = cpc; }
    }
    return best;
}

// Launch geometry of the fused step for this species' current state; rows == 0 when a cell may not fit
// a tile.  A tile must hold at least one cell; maxcount is the bound read at the last sync, so leave room
// for it to grow.
static FusedGeom fused_geom(const pic_species *s)
{
    const pic_sim *sim = s->sim;
    FusedGeom g{};
    // Largest cell a tile must hold: the largest count last seen (telemetry lags a few steps: leave 1/16 + 8), and
    // never less than the expected maximum of nc Poisson counts of the mean occupancy -- a state that starts with
    // exactly equal counts (the configs do) reaches that within a few steps.
    const int mc = std::max(s->h_maxcount, 1);
    const double mean = (double)s->n_ub / (double)sim->nc;
    const int poisson_max = (int)std::ceil(mean + std::sqrt(2.0 * mean * std::log((double)sim->nc + 1.0)));
    const int top = std::max(mc, poisson_max);
    const int need = top + top / 16 + 8 + 2;
    g.rows = sim->opt_fused_rows;
    if (g.rows == 0) g.rows = need <= 8 * 32 ? 8 : need <= 12 * 32 ? 12 : need <= 16 * 32 ? 16 : 0;
    if (g.rows == 0) return g;
    // two stages under the 8-row tiles (11 CTAs of 19.7 KB per SM: measured 3-7 % faster than one stage at 16 CTAs);
    // the wider tiles keep one stage (a second one would halve their CTAs per SM: measured slower)
    g.stages = !sim->opt_fused_tma ? 0 : (sim->opt_fused_stages ? sim->opt_fused_stages : (g.rows == 8 ? 2 : 1));
    // queue of the right-movers that wait for the next tile: the usual one until a step has overflowed it
    g.def = s->h_maxdef > FUSED_DEF ? FUSED_DEF_BIG : FUSED_DEF;
    if (!sim->opt_fused_tma) g.def = FUSED_DEF; // the plain-load A/B variant exists with the usual queue only
    g.cpc = fused_cells_per_cta(s, g.rows, g.stages, g.def, &g.taper);
    g.slots = sim->opt_fused_slots ? std::min(sim->opt_fused_slots, g.rows * 32) : g.rows * 32;
    g.smem = (size_t)fused_layout(g.rows * 32, g.cpc, g.stages, g.def).total;
    g.ctas_per_sm = fused_ctas_per_sm(g.rows, g.cpc, g.stages, g.def);
    return g;
}

static int fused_rows(const pic_species *s, int *ctas_per_sm)
{
    const FusedGeom g = fused_geom(s);
    if (g.rows && ctas_per_sm) *ctas_per_sm = g.ctas_per_sm;
    return g.rows;
}

// Chunk schedule of one fused launch (FusedArgs::seg_*): the bulk of the grid in chunks of cpc cells, then -- `taper`
// times -- one machine-load (sm_count * ctas_per_sm CTAs) of chunks half as large as the ones before, the smallest
// last.  CTAs start in blockIdx order, so the CTAs still running when the grid drains are the short ones: the tail in
// which SMs idle shrinks with the chunk size while the bulk pays the halo cells of large chunks only.  Returns the grid.
static int fused_schedule(FusedArgs &a, int nc, int cpc, int taper, int resident)
{
    int sizes[FUSED_SEGS], cells[FUSED_SEGS];
    int nseg = 1, left = nc;
    sizes[0] = cpc;
    for (int t = 1; t <= taper && nseg < FUSED_SEGS; ++t) {
        const int sz = cpc >> t;
        if (sz < 2) break;
        sizes[nseg++] = sz;
    }
    for (int sg = nseg - 1; sg >= 1; --sg) { // the tail segments take their cells from the end of the grid
        const long long want = (long long)resident * sizes[sg];
        cells[sg] = (int)std::min<long long>(want, std::max(0, left - cpc)); // the bulk keeps at least one chunk
        left -= cells[sg];
    }
    cells[0] = left;
    int blk = 0, cell = 0;
    for (int sg = 0; sg < FUSED_SEGS; ++sg) {
        if (sg < nseg && cells[sg] > 0) {
            a.seg_blk[sg] = blk; a.seg_cell[sg] = cell; a.seg_cpc[sg] = sizes[sg];
            blk += (cells[sg] + sizes[sg] - 1) / sizes[sg];
            cell += cells[sg];
        } else { // empty segment: no CTA selects it
            a.seg_blk[sg] = sg == 0 ? 0 : INT_MAX; a.seg_cell[sg] = cell; a.seg_cpc[sg] = sizes[0];
        }
        a.seg_cell[sg + 1] = cell;
    }
    return blk;
}

// One fused push+arrange step.  Nothing is enqueued behind it to catch a declined step: the device records
// the first step that declined and turns every later fused launch into a no-op, and verify_fused() -- run by
// every synchronising call and before any non-fused work -- rewinds the host bookkeeping to that step and
// redoes the rest with the split kernels.
static int push_fused(pic_species *s)
{
    pic_sim *sim = s->sim;
    if (s->tel_pending) { // has a telemetry copy landed?  (never waits)
        const cudaError_t q = cudaEventQuery(s->tel_ev);
        if (q == cudaSuccess) {
            s->tel_pending = false;
            if (!s->h_tel->fused_disabled) s->h_maxcount = s->h_tel->maxcount;
        } else if (q == cudaErrorNotReady) {
            cudaGetLastError(); // not an error: clear it so that the launch checks below do not see it
        } else {
            return cuda_fail(q, "cudaEventQuery telemetry");
        }
    }
    const int src = s->cur, dst = s->cur ^ 1;
    const int oo = s->cur_off, on = s->cur_off ^ 1;
    FusedArgs a{};
    a.sx = s->x[src]; a.svx = s->vx[src]; a.svy = s->vy[src]; a.svz = s->vz[src];
    a.dx = s->x[dst]; a.dvx = s->vx[dst]; a.dvy = s->vy[dst]; a.dvz = s->vz[dst]; a.dcell = s->cell[dst];
    a.E = sim->d_E;
    a.off_old = s->d_off[oo];
    a.count_new = s->d_count[on]; a.off_new = s->d_off[on];
    a.st = s->d_st;
    a.k = s->k;
    a.capacity = s->capacity;
    const FusedGeom geo = fused_geom(s);
    a.CPC = geo.cpc;
    a.SCAP = geo.slots;
    a.NST = geo.stages;
    {   // PIC_TRACE: report the launch geometry whenever it changes
        static const bool trace = getenv("PIC_TRACE") != nullptr;
        int *last = s->trace_last; // per species: sims of different threads share no mutable static
        const int now[6] = {geo.rows, geo.cpc + 1000 * geo.taper, geo.stages, geo.def, geo.ctas_per_sm, (int)geo.smem};
        if (trace && memcmp(last, now, sizeof now)) {
            memcpy(last, now, sizeof now);
            fprintf(stderr, "[pic fused] step %lld: rows %d, cells/CTA %d (taper %d), stages %d, queue %d, CTAs/SM %d, smem %d B (maxcount %d, maxdef %d)\n",
                    s->steps, geo.rows, geo.cpc, geo.taper, geo.stages, geo.def, geo.ctas_per_sm, (int)geo.smem, s->h_maxcount, s->h_maxdef);
        }
    }
    a.step_id = (int)(s->steps & 0x7fffffff);
    a.frozen = sim->in_cycle ? sim->d_frozen : nullptr;
    const int rows = geo.rows;
    const int grid = fused_schedule(a, sim->nc, a.CPC, geo.taper, sim->sm_count * geo.ctas_per_sm);
    const size_t smem = geo.smem;
    if (s->unv_steps == 0) {
        s->unv_steps0 = s->steps;
        s->unv_cur0 = s->cur;
        s->unv_off0 = s->cur_off;
    }
    {
        KernelSpan span(sim, K_FUSED, s->stream);
        // programmatic dependent launches (option "fused_pdl"): each kernel of the chain edge -> streaming -> commit ->
        // next step's edge is set up while its predecessor still runs and waits (griddepcontrol.wait) for it before it
        // reads or writes anything the predecessor touches; the streaming kernel's prologue overlaps the edge kernel
        auto launch = [&](bool pdl, auto kern, int grid, int block, size_t smem, auto... args) -> cudaError_t {
            if (!pdl) {
                kern<<<grid, block, smem, s->stream>>>(args...);
                return cudaSuccess;
            }
            cudaLaunchConfig_t cfg{};
            cfg.gridDim = dim3((unsigned)grid);
            cfg.blockDim = dim3((unsigned)block);
            cfg.dynamicSmemBytes = smem;
            cfg.stream = s->stream;
            cudaLaunchAttribute attr[1];
            attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
            attr[0].val.programmaticStreamSerializationAllowed = 1;
            cfg.attrs = attr;
            cfg.numAttrs = 1;
            return cudaLaunchKernelEx(&cfg, kern, args...);
        };
        // The edge kernel only when the last kernel this library launched was this species' previous commit kernel
        // (which waited for its step to complete and triggers nothing early): behind any other kernel the streaming
        // kernel's prologue -- it starts with the edge kernel and reads E, offsets and particles before it waits --
        // could run before that kernel's writes are visible.
        const bool pdl = sim->opt_fused_pdl != 0;
        const bool chained = pdl && s->chain_valid && s->chain_mark == sim->launches;
        CU(launch(chained, fused_edge_kernel, 1, 128, (size_t)0, a));
        if (int rc = launch_check(sim, "fused_edge_kernel")) return rc;
        const bool bz0 = s->k.tz == 0.0 && s->k.sz == 0.0; // B in the x-y plane: the kernel drops the exact-zero products
        void (*kern)(FusedArgs) = fused_pick(rows, sim->periodic != 0, bz0, sim->opt_fused_tma != 0, geo.def);
        CU(launch(pdl, kern, grid, 32, smem, a));
        if (int rc = launch_check(sim, "fused_kernel")) return rc;
        CU(launch(pdl, fused_commit_kernel, 1, 1, (size_t)0, s->d_st, a.step_id, a.frozen));
        if (int rc = launch_check(sim, "fused_commit_kernel")) return rc;
        s->chain_valid = true;
        s->chain_mark = sim->launches;
    }
    if (++s->tel_step >= FUSED_TELEMETRY_STEPS && !s->tel_pending) {
        CU(cudaMemcpyAsync(s->h_tel, s->d_st, sizeof(DevState), cudaMemcpyDeviceToHost, s->stream));
        CU(cudaEventRecord(s->tel_ev, s->stream));
        s->tel_pending = true;
        s->tel_step = 0;
    }
    s->unv_steps++;
    s->h_steps_since_sync++;
    // a step enqueued while max |E| of a device-side field is still unknown has no known kick: the bound stays
    // "unknown" (infinite) until the next read_state refreshes the speed bound, even if pic_set_field intervenes
    s->h_kick_acc += s->sim->emax_known ? s->vkick : (double)INFINITY;
    s->cur = dst;
    s->cur_off = on;
    s->counts_fresh = true;
    s->all_live = true;
    s->reset_w = true;
    s->h_wsum = 0;
    s->h_grouped = true;
    return PIC_OK;
}

// Check the fused steps enqueued since the last check.  If one declined, the device state is the one before
// that step (later fused launches did nothing): rewind the host bookkeeping to it and redo the remaining steps
// through the split path.  Syncs when there is anything to check.
static int verify_fused(pic_species *s)
{
    if (!s->sim->cyc_pending.empty()) return verify_cycles(s->sim); // unchecked pic_cycle work: all species together
    if (s->unv_steps == 0) return PIC_OK;
    DevState h;
    CU(cudaMemcpyAsync(&h, s->d_st, sizeof h, cudaMemcpyDeviceToHost, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    const long long run = s->unv_steps;
    s->unv_steps = 0;
    if (!h.fused_disabled) return PIC_OK;
    s->fused_off = true;
    s->declined_at = s->unv_steps0 + run;
    const long long k = ((long long)h.fail_step - (s->unv_steps0 & 0x7fffffff)) & 0x7fffffff; // steps that completed
    if (k >= run) {
        snprintf(g_err, sizeof g_err, "fused step bookkeeping: declined step %d outside the unverified run", h.fail_step);
        return PIC_ESTATE;
    }
    s->cur = s->unv_cur0 ^ (int)(k & 1);
    s->cur_off = s->unv_off0 ^ (int)(k & 1);
    s->steps = s->unv_steps0 + k;
    s->counts_fresh = true;
    s->all_live = true;
    s->reset_w = true;
    s->h_wsum = 0;
    s->h_grouped = true;
    s->h_vmax = std::sqrt((double)bits_to_float(h.vmax2));
    s->h_steps_since_sync = 0;
    s->h_kick_acc = 0;
    s->h_maxcount = h.maxcount;
    s->h_maxdef = std::max(s->h_maxdef, h.maxdef);
    for (long long left = run - k; left > 0;) {
        const int chunk = (int)std::min<long long>(left, 1 << 20);
        if (int rc = pic_push(s, chunk)) return rc;
        left -= chunk;
    }
    return PIC_OK;
}

extern "C" int pic_push(pic_species *s, int nsteps)
{
    if (!s || nsteps < 0) return PIC_EINVAL;
    if (!s->sim->in_cycle && !s->sim->cyc_pending.empty()) // unchecked pic_cycle work: settle it before stepping on
        if (int rc = verify_cycles(s->sim)) return rc;
    for (int it = 0; it < nsteps; ++it) {
        const bool will_arrange = s->arrange_every > 0 && ((s->steps + 1) % s->arrange_every) == 0;
        const bool fused = will_arrange && fused_possible(s) && s->counts_fresh && s->all_live && s->n_ub > 0;
        if (fused) {
            if (int rc = push_fused(s)) return rc;
            s->steps++;
            continue;
        }
        if (int rc = verify_fused(s)) return rc; // the split kernels need the true state (total step count unchanged)
        if (int rc = push_split(s, will_arrange)) return rc;
        s->steps++;
        if (will_arrange)
            if (int rc = arrange_split(s, true, true)) return rc;
    }
    return PIC_OK;
}

// ------------------------------------------------------------------------------------------
// read-outs
// ------------------------------------------------------------------------------------------
static int read_state(pic_species *s, DevState &h)
{
    if (int rc = verify_fused(s)) return rc;
    CU(cudaMemcpyAsync(&h, s->d_st, sizeof h, cudaMemcpyDeviceToHost, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    if (h.n >= 0 && h.n <= s->n_ub) s->n_ub = h.n;
    s->h_vmax = std::sqrt((double)bits_to_float(h.vmax2));
    s->h_steps_since_sync = 0;
    s->h_kick_acc = 0;
    if (!s->sim->emax_known) { // the field was replaced on the device: fetch its max |E| for the displacement bound
        pic_sim *sim = s->sim;
        unsigned long long bits = 0;
        CU(cudaMemcpyAsync(&bits, sim->d_emax, sizeof bits, cudaMemcpyDeviceToHost, s->stream));
        CU(cudaStreamSynchronize(s->stream));
        double em;
        memcpy(&em, &bits, sizeof em);
        sim->Emax = em;
        sim->emax_known = true;
        for (pic_species *o : sim->sp) o->vkick = 2.0 * std::fabs(o->k.h) * em;
    }
    if (h.fused_disabled) s->fused_off = true;
    s->h_maxcount = h.maxcount;
    s->h_maxdef = std::max(s->h_maxdef, h.maxdef);
    s->h_abort_reason = h.abort_reason;
    // A declined fused path comes back once the cause is gone: the state is arranged, the split mover's last
    // step moved no particle by more than one cell, and some steps have passed since the decline.
    if (s->fused_off && s->arrange_every == 1 && s->counts_fresh && h.w_acc <= 1 && h.status == 0 &&
        s->steps - s->declined_at >= FUSED_RETRY_STEPS && !(h.abort_reason & FA_EDGE_OVERFLOW) && s->h_maxdef <= FUSED_DEF_BIG) {
        const int zero = 0;
        CU(cudaMemcpyAsync(&s->d_st->fused_disabled, &zero, sizeof zero, cudaMemcpyHostToDevice, s->stream));
        CU(cudaStreamSynchronize(s->stream));
        s->fused_off = false;
    }
    return PIC_OK;
}

// All species of the sim, nsteps steps each.  The species are independent within a step (they share only the field,
// read-only), so each runs on a stream of its own for the duration of the call: their kernels overlap, in particular
// the ramp and the tail of one species' grid with the bulk of another's ("two streams on one
// GPU").  Fork and join are events: on return everything is ordered on the sim's stream again.
extern "C" int pic_push_all(pic_sim *sim, int nsteps)
{
    if (!sim || nsteps < 0) return PIC_EINVAL;
    NvtxRange range("pic_push_all");
    // Unchecked pic_cycle work is settled HERE, while every species still runs on the sim's stream: should a fused step
    // of those cycles have declined, verify_cycles redoes pushes, depositions (species after species into one rho)
    // and field solves, which are ordered only on a common stream.  Left to the first pic_push below, that redo
    // would run with each species on its own, mutually unordered stream.
    if (!sim->in_cycle && !sim->cyc_pending.empty())
        if (int rc = verify_cycles(sim)) return rc;
    const size_t ns = sim->sp.size();
    if (ns <= 1 || !sim->opt_species_streams) {
        for (int it = 0; it < nsteps; ++it)
            for (pic_species *s : sim->sp)
                if (int rc = pic_push(s, 1)) return rc;
        return PIC_OK;
    }
    if (!sim->fork_ev) CU(cudaEventCreateWithFlags(&sim->fork_ev, cudaEventDisableTiming));
    for (pic_species *s : sim->sp) {
        if (!s->own_stream) CU(cudaStreamCreateWithFlags(&s->own_stream, cudaStreamNonBlocking));
        if (!s->join_ev) CU(cudaEventCreateWithFlags(&s->join_ev, cudaEventDisableTiming));
    }
    CU(cudaEventRecord(sim->fork_ev, sim->stream));
    int rc = PIC_OK;
    for (pic_species *s : sim->sp) { // fork; a failure still goes through the join below, which restores every stream
        const cudaError_t e = cudaStreamWaitEvent(s->own_stream, sim->fork_ev, 0);
        if (e != cudaSuccess) { rc = cuda_fail(e, "pic_push_all fork"); break; }
        s->stream = s->own_stream;
    }
    for (int it = 0; it < nsteps && rc == PIC_OK; ++it)
        for (pic_species *s : sim->sp) {
            const unsigned long long before = sim->launches;
            if ((rc = pic_push(s, 1)) != PIC_OK) break;
            // these launches went to this species' own stream: they do not stand between another species' commit
            // kernel and its next edge kernel (push_fused: chain_mark)
            for (pic_species *o : sim->sp)
                if (o != s) o->chain_mark += sim->launches - before;
        }
    for (pic_species *s : sim->sp) { // join, whatever happened
        if (s->stream != s->own_stream) continue; // the fork failed before this species
        s->stream = sim->stream;
        const cudaError_t e1 = cudaEventRecord(s->join_ev, s->own_stream);
        const cudaError_t e2 = e1 == cudaSuccess ? cudaStreamWaitEvent(sim->stream, s->join_ev, 0) : e1;
        if (e2 != cudaSuccess && rc == PIC_OK) rc = cuda_fail(e2, "pic_push_all join");
    }
    return rc;
}

extern "C" int pic_wall_flux(pic_species *s, pic_wall_flux_t *out)
{
    if (!s || !out) return PIC_EINVAL;
    DevState h;
    if (int rc = read_state(s, h)) return rc;
    out->left_total = h.wall[0];
    out->right_total = h.wall[1];
    out->left_recent = h.wall[0] - s->wall_last[0];
    out->right_recent = h.wall[1] - s->wall_last[1];
    out->steps_total = (uint64_t)s->steps;
    out->steps_recent = (uint64_t)(s->steps - s->steps_at_last_flux);
    s->wall_last[0] = h.wall[0];
    s->wall_last[1] = h.wall[1];
    s->steps_at_last_flux = s->steps;
    return status_to_rc(h.status);
}

extern "C" int pic_n_slots(pic_species *s, int64_t *n)
{
    if (!s || !n) return PIC_EINVAL;
    DevState h;
    if (int rc = read_state(s, h)) return rc;
    *n = h.n;
    return status_to_rc(h.status);
}

extern "C" int pic_n_live(pic_species *s, int64_t *n)
{
    if (!s || !n) return PIC_EINVAL;
    DevState h;
    if (int rc = read_state(s, h)) return rc;
    // slots in use minus the particles absorbed (flagged, still in place) since the last arrange
    *n = (int64_t)h.n - (int64_t)((h.wall[0] + h.wall[1]) - h.wall_arr);
    return status_to_rc(h.status);
}

extern "C" int pic_active_buffer(pic_species *s, int *which)
{
    if (!s || !which) return PIC_EINVAL;
    if (int rc = verify_fused(s)) return rc;
    *which = s->cur;
    return PIC_OK;
}

extern "C" int pic_step_count(pic_species *s, int64_t *steps)
{
    if (!s || !steps) return PIC_EINVAL;
    *steps = s->steps;
    return PIC_OK;
}

extern "C" int pic_cell_counts(pic_species *s, int32_t *count_host, int32_t *offset_host)
{
    if (!s) return PIC_EINVAL;
    if (int rc = verify_fused(s)) return rc;
    if (!s->counts_fresh) return PIC_ESTATE;
    const int nc = s->sim->nc;
    if (count_host)
        CU(cudaMemcpyAsync(count_host, s->d_count[s->cur_off], sizeof(int) * (size_t)nc, cudaMemcpyDeviceToHost, s->stream));
    if (offset_host)
        CU(cudaMemcpyAsync(offset_host, s->d_off[s->cur_off], sizeof(int) * ((size_t)nc + 1), cudaMemcpyDeviceToHost, s->stream));
    CU(cudaStreamSynchronize(s->stream));
    return PIC_OK;
}

static int deposit_enqueue(pic_species *s, double weight, double *rho_dev, int accumulate);

extern "C" int pic_deposit(pic_species *s, double weight, double *rho_dev, int accumulate)
{
    if (!s || !rho_dev || !std::isfinite(weight)) return PIC_EINVAL;
    if (int rc = verify_fused(s)) return rc;
    if (!s->counts_fresh || !s->all_live) return PIC_ESTATE;
    return deposit_enqueue(s, weight, rho_dev, accumulate);
}

// The two deposition kernels, enqueued without any host-side check (the state must be arranged and all live).
static int deposit_enqueue(pic_species *s, double weight, double *rho_dev, int accumulate)
{
    pic_sim *sim = s->sim;
    const int nc = sim->nc;
    if (!s->d_cs) {
        cudaError_t e = dev_alloc(&s->d_cs, sizeof(double2) * (size_t)nc, sim->device, s->stream);
        if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? PIC_ENOMEM : cuda_fail(e, "cudaMalloc deposition sums");
    }
    DepositArgs a{};
    a.x = s->x[s->cur];
    a.off = s->d_off[s->cur_off];
    a.cs = s->d_cs;
    a.nc = nc;
    a.inv_dx = s->k.inv_dx;
    KernelSpan span(sim, K_DEPOSIT, s->stream);
    const int lpc = s->n_ub <= 448LL * nc ? 16 : 32; // lanes per cell from the mean particles per cell (16 measured best up to 200)
    const long long threads = (long long)nc * lpc;
    const unsigned blocks = (unsigned)((threads + DEP_THREADS - 1) / DEP_THREADS);
    if (lpc == 16) deposit_cell_kernel<16><<<blocks, DEP_THREADS, 0, s->stream>>>(a);
    else deposit_cell_kernel<32><<<blocks, DEP_THREADS, 0, s->stream>>>(a);
    if (int rc = launch_check(sim, "deposit_cell_kernel")) return rc;
    deposit_node_kernel<<<(nc + 1 + 255) / 256, 256, 0, s->stream>>>(s->d_cs, nc, sim->periodic, weight, accumulate ? 1 : 0, rho_dev);
    return launch_check(sim, "deposit_node_kernel");
}


// ------------------------------------------------------------------------------------------
// pic_cycle: the closed PIC cycle, enqueued without a host round trip
// ------------------------------------------------------------------------------------------
// A fused step is checked on the device and may decline (fused.cuh); pic_deposit and pic_solve_field therefore check
// the unverified steps first, which synchronises once per cycle.  pic_cycle owns the whole loop instead, so it can
// replay it: steps (every species on its own stream), depositions and field solves are enqueued unchecked; should a
// step decline, the device freezes -- that species' commit kernel raises the sim's flag, no species starts another
// fused step, field_e_kernel leaves E alone (the depositions and the rest of the solve only write scratch and rho) --
// and the next synchronising call finds, per species, the last step that completed, and redoes every cycle from the
// first incomplete one with the ordinary checked calls.  Results are those of the checked loop either way.
static bool cycle_fast_ok(pic_sim *sim)
{
    if (sim->nc < 2 || !sim->opt_cycle_async) return false;
    for (pic_species *s : sim->sp)
        if (!(s->arrange_every == 1 && fused_possible(s) && s->counts_fresh && s->all_live && s->n_ub > 0)) return false;
    return true;
}

static int verify_cycles(pic_sim *sim)
{
    if (sim->cyc_pending.empty()) return PIC_OK;
    std::vector<pic_sim::CycleRec> recs;
    recs.swap(sim->cyc_pending); // from here on the ordinary, checked calls can be used
    long long total = 0;
    for (const auto &r : recs) total += r.ncycles;
    const size_t ns = sim->sp.size();
    std::vector<DevState> h(ns);
    for (size_t i = 0; i < ns; ++i)
        CU(cudaMemcpyAsync(&h[i], sim->sp[i]->d_st, sizeof(DevState), cudaMemcpyDeviceToHost, sim->stream));
    CU(cudaStreamSynchronize(sim->stream));
    bool any = false;
    long long first = total; // the first cycle whose step some species did not complete
    for (size_t i = 0; i < ns; ++i) {
        pic_species *s = sim->sp[i];
        const long long run = s->unv_steps;
        s->unv_steps = 0;
        if (run != total) {
            snprintf(g_err, sizeof g_err, "pic_cycle bookkeeping: %lld unverified steps against %lld pending cycles", run, total);
            return PIC_ESTATE;
        }
        if (!h[i].fused_disabled) continue; // completed every step
        any = true;
        const long long k = ((long long)h[i].fail_step - (s->unv_steps0 & 0x7fffffff)) & 0x7fffffff; // steps that completed
        if (k >= run) {
            snprintf(g_err, sizeof g_err, "pic_cycle bookkeeping: declined step %d outside the pending cycles", h[i].fail_step);
            return PIC_ESTATE;
        }
        first = std::min(first, k);
        s->fused_off = true;
        s->declined_at = s->unv_steps0 + run;
        s->cur = s->unv_cur0 ^ (int)(k & 1);
        s->cur_off = s->unv_off0 ^ (int)(k & 1);
        s->steps = s->unv_steps0 + k;
        s->counts_fresh = true;
        s->all_live = true;
        s->reset_w = true;
        s->h_wsum = 0;
        s->h_grouped = true;
        s->h_vmax = std::sqrt((double)bits_to_float(h[i].vmax2));
        s->h_steps_since_sync = 0;
        s->h_kick_acc = 0;
        s->h_maxcount = h[i].maxcount;
        s->h_maxdef = std::max(s->h_maxdef, h[i].maxdef);
        s->chain_valid = false;
    }
    if (!any) return PIC_OK;
    CU(cudaMemsetAsync(sim->d_frozen, 0, sizeof(int), sim->stream));
    {   // the field in force is the one the frozen device kept; its max |E| was cleared by the solves that were skipped
        CU(cudaMemsetAsync(sim->d_emax, 0, sizeof(unsigned long long), sim->stream));
        field_emax_kernel<<<(sim->nc + 1 + FLD_THREADS - 1) / FLD_THREADS, FLD_THREADS, 0, sim->stream>>>(sim->d_E, sim->nc, sim->d_emax);
        if (int rc = launch_check(sim, "field_emax_kernel")) return rc;
        sim->emax_known = false;
    }
    long long idx = 0;
    for (const auto &r : recs)
        for (int c = 0; c < r.ncycles; ++c, ++idx) {
            if (idx < first) continue;
            for (pic_species *s : sim->sp) // a species that ran concurrently may have completed this cycle's step
                if (s->steps < s->cyc_step0 + idx + 1)
                    if (int rc = pic_push(s, 1)) return rc;
            for (size_t i = 0; i < ns; ++i)
                if (int rc = pic_deposit(sim->sp[i], r.w[i], r.rho, i > 0)) return rc;
            if (int rc = pic_solve_field(sim, r.rho, r.passes, r.phi)) return rc;
        }
    return PIC_OK;
}

extern "C" int pic_cycle(pic_sim *sim, int ncycles, const double *weights, int smooth_passes, double *rho_dev, double *phi_dev)
{
    if (!sim || ncycles < 0 || !weights || !rho_dev || smooth_passes < 0 || smooth_passes > 1024) return PIC_EINVAL;
    if (sim->nc < 2) return PIC_EINVAL;
    NvtxRange range("pic_cycle");
    const size_t ns = sim->sp.size();
    for (size_t i = 0; i < ns; ++i)
        if (!std::isfinite(weights[i])) return PIC_EINVAL;
    for (int c = 0; c < ncycles; ++c) {
        if (sim->cyc_pending.empty())
            for (pic_species *s : sim->sp) // fused steps of earlier plain pic_push calls: check them first
                if (int rc = verify_fused(s)) return rc;
        if (!cycle_fast_ok(sim)) { // the ordinary checked calls
            if (int rc = verify_cycles(sim)) return rc;
            if (int rc = pic_push_all(sim, 1)) return rc;
            for (size_t i = 0; i < ns; ++i)
                if (int rc = pic_deposit(sim->sp[i], weights[i], rho_dev, i > 0)) return rc;
            if (int rc = pic_solve_field(sim, rho_dev, smooth_passes, phi_dev)) return rc;
            continue;
        }
        if (sim->cyc_pending.empty()) {
            if (!sim->d_frozen) {
                cudaError_t e = dev_alloc(&sim->d_frozen, sizeof(int), sim->device, sim->stream);
                if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? PIC_ENOMEM : cuda_fail(e, "cudaMalloc cycle flag");
                CU(cudaMemsetAsync(sim->d_frozen, 0, sizeof(int), sim->stream));
            }
            for (pic_species *s : sim->sp) s->cyc_step0 = s->steps;
        }
        sim->in_cycle = true;
        const int rc_push = pic_push_all(sim, 1);
        sim->in_cycle = false;
        if (rc_push) return rc_push;
        // recorded before the rest is enqueued: from here on a synchronising call must find (and can redo) this cycle
        pic_sim::CycleRec *last = sim->cyc_pending.empty() ? nullptr : &sim->cyc_pending.back();
        if (last && last->passes == smooth_passes && last->rho == rho_dev && last->phi == phi_dev &&
            std::equal(last->w.begin(), last->w.end(), weights))
            last->ncycles++;
        else
            sim->cyc_pending.push_back({1, std::vector<double>(weights, weights + ns), smooth_passes, rho_dev, phi_dev});
        for (size_t i = 0; i < ns; ++i)
            if (int rc = deposit_enqueue(sim->sp[i], weights[i], rho_dev, i > 0)) return rc;
        if (int rc = solve_enqueue(sim, rho_dev, smooth_passes, phi_dev, sim->d_frozen)) return rc;
    }
    return PIC_OK;
}

extern "C" int pic_arrange_info(pic_species *s, int32_t *w_bound, int32_t *used_general)
{
    if (!s) return PIC_EINVAL;
    DevState h;
    if (int rc = read_state(s, h)) return rc;
    if (w_bound) *w_bound = h.w_acc;
    if (used_general) *used_general = h.used_general;
    return PIC_OK;
}

extern "C" int pic_fused_info(pic_species *s, int32_t *active, int32_t *decline_reasons, int32_t *stage_slots,
                              int32_t *ctas_per_sm)
{
    if (!s) return PIC_EINVAL;
    DevState h;
    if (int rc = read_state(s, h)) return rc;
    if (active) *active = fused_possible(s) ? 1 : 0;
    if (decline_reasons) *decline_reasons = h.abort_reason;
    int ctas = 0;
    const int cap = fused_rows(s, &ctas) ? fused_geom(s).slots : 0;
    if (stage_slots) *stage_slots = cap;
    if (ctas_per_sm) *ctas_per_sm = ctas;
    return PIC_OK;
}

extern "C" int pic_sync(pic_sim *sim)
{
    if (!sim) return PIC_EINVAL;
    CU(cudaStreamSynchronize(sim->stream));
    int rc = PIC_OK;
    for (pic_species *s : sim->sp) {
        DevState h;
        if (int r = read_state(s, h)) return r;
        if (int r = status_to_rc(h.status)) rc = r;
    }
    return rc;
}

// ------------------------------------------------------------------------------------------
// end-to-end call with host buffers
// ------------------------------------------------------------------------------------------
extern "C" int pic_run_host(const pic_grid_desc *g, pic_host_species *hs, int nspecies, int nsteps)
{
    if (!g || !hs || nspecies < 1 || nsteps < 0) return PIC_EINVAL;
    NvtxRange range("pic_run_host");
    cudaStream_t stream = static_cast<cudaStream_t>(g->stream);
    // optional wall-clock trace of the phases (stderr), switched on by the environment variable PIC_TRACE
    const bool trace = getenv("PIC_TRACE") != nullptr;
    const auto t_begin = std::chrono::steady_clock::now();
    auto mark = [&](const char *what) {
        if (!trace) return;
        cudaStreamSynchronize(stream);
        const double ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_begin).count();
        fprintf(stderr, "[pic_run_host] %-28s %9.3f ms\n", what, ms);
    };
    std::vector<pic_species_desc> descs(nspecies);
    int rc = PIC_OK;
    pic_sim *sim = nullptr;
    char *arena = nullptr;
    bool arena_cached = false;
    int arena_device = -1;
    cudaStream_t copy_stream = nullptr;
    auto align256 = [](size_t b) { return (b + 255) & ~(size_t)255; };
    do {
        // one device allocation for everything: two buffer sets and the workspace of every species
        size_t total = 0;
        for (int i = 0; i < nspecies; ++i) {
            const pic_host_species &h = hs[i];
            if (h.n < 0 || (h.n > 0 && (!h.x || !h.vx || !h.vy || !h.vz || !h.cell))) { rc = PIC_EINVAL; break; }
            const size_t nb = align256(sizeof(double) * (size_t)h.n + 16), ni = align256(sizeof(int32_t) * (size_t)h.n + 16);
            total += 2 * (4 * nb + ni) + align256(pic_workspace_bytes(g->nc, h.n) + 16);
        }
        if (rc) break;
        int device = 0;
        cudaGetDevice(&device);
        cudaError_t e = cudaSuccess;
        {   // the previous call's arena if it is large enough and free (a concurrent call of another thread gets its own)
            std::lock_guard<std::mutex> lock(g_mem_mu);
            if (device >= 0 && device < 64 && !g_arena[device].in_use) {
                if (g_arena[device].p && g_arena[device].bytes < total) {
                    cudaFree(g_arena[device].p);
                    g_arena[device].p = nullptr;
                    g_arena[device].bytes = 0;
                }
                if (!g_arena[device].p) {
                    e = cudaMalloc(&g_arena[device].p, total ? total : 256);
                    if (e != cudaSuccess) g_arena[device].p = nullptr;
                    else g_arena[device].bytes = total ? total : 256;
                }
                if (g_arena[device].p) {
                    arena = g_arena[device].p;
                    g_arena[device].in_use = true;
                    arena_cached = true;
                    arena_device = device;
                }
            }
        }
        if (!arena && e == cudaSuccess) e = cudaMalloc(&arena, total ? total : 256);
        if (e != cudaSuccess || !arena) { cudaGetLastError(); arena = nullptr; rc = PIC_ENOMEM; break; }
        mark("device arena allocated");
        size_t off = 0;
        auto carve = [&](size_t bytes) { void *p = arena + off; off += bytes; return p; };
        for (int i = 0; i < nspecies; ++i) {
            pic_host_species &h = hs[i];
            pic_species_desc &d = descs[i];
            memset(&d, 0, sizeof d);
            d.qm = h.qm; d.n = h.n; d.capacity = h.n; d.arrange_every = h.arrange_every;
            const size_t nb = align256(sizeof(double) * (size_t)h.n + 16), ni = align256(sizeof(int32_t) * (size_t)h.n + 16);
            for (int b = 0; b < 2; ++b) {
                d.x[b] = (double *)carve(nb); d.vx[b] = (double *)carve(nb);
                d.vy[b] = (double *)carve(nb); d.vz[b] = (double *)carve(nb);
                d.cell[b] = (int32_t *)carve(ni);
            }
            d.workspace_bytes = pic_workspace_bytes(g->nc, h.n);
            d.workspace = carve(align256(d.workspace_bytes + 16));
            const size_t cb = sizeof(double) * (size_t)h.n, ci = sizeof(int32_t) * (size_t)h.n;
            if (h.n > 0) {
                e = cudaMemcpyAsync(d.x[0], h.x, cb, cudaMemcpyHostToDevice, stream);
                if (e == cudaSuccess) e = cudaMemcpyAsync(d.cell[0], h.cell, ci, cudaMemcpyHostToDevice, stream);
                if (e == cudaSuccess) e = cudaMemcpyAsync(d.vx[0], h.vx, cb, cudaMemcpyHostToDevice, stream);
                if (e == cudaSuccess) e = cudaMemcpyAsync(d.vy[0], h.vy, cb, cudaMemcpyHostToDevice, stream);
                if (e == cudaSuccess) e = cudaMemcpyAsync(d.vz[0], h.vz, cb, cudaMemcpyHostToDevice, stream);
            }
            if (e != cudaSuccess) { rc = cuda_fail(e, "cudaMemcpyAsync H2D"); break; }
        }
        if (rc) break;
        mark("H2D done");
        rc = pic_create(g, descs.data(), nspecies, &sim);
        if (rc) break;
        mark("pic_create done");
        rc = pic_push_all(sim, nsteps);
        if (rc) break;
        mark("steps done");
        // the copies back: each array on a second stream as soon as its species has been read out, so that they
        // queue behind one another without host round trips
        if (cudaStreamCreateWithFlags(&copy_stream, cudaStreamNonBlocking) != cudaSuccess) { rc = cuda_fail(cudaGetLastError(), "copy stream"); break; }
        for (int i = 0; i < nspecies && rc == PIC_OK; ++i) {
            pic_species *s = sim->sp[i];
            pic_host_species &h = hs[i];
            pic_wall_flux_t wf;
            rc = pic_wall_flux(s, &wf); // syncs: the species' state is final
            if (rc) break;
            int64_t n = 0;
            rc = pic_n_slots(s, &n);
            if (rc) break;
            h.n_out = n; h.wall_left = wf.left_total; h.wall_right = wf.right_total;
            const size_t nb = sizeof(double) * (size_t)n, ni = sizeof(int32_t) * (size_t)n;
            const int b = s->cur;
            e = cudaSuccess;
            if (n > 0) {
                e = cudaMemcpyAsync(h.x, s->x[b], nb, cudaMemcpyDeviceToHost, copy_stream);
                if (e == cudaSuccess) e = cudaMemcpyAsync(h.vx, s->vx[b], nb, cudaMemcpyDeviceToHost, copy_stream);
                if (e == cudaSuccess) e = cudaMemcpyAsync(h.vy, s->vy[b], nb, cudaMemcpyDeviceToHost, copy_stream);
                if (e == cudaSuccess) e = cudaMemcpyAsync(h.vz, s->vz[b], nb, cudaMemcpyDeviceToHost, copy_stream);
                if (e == cudaSuccess) e = cudaMemcpyAsync(h.cell, s->cell[b], ni, cudaMemcpyDeviceToHost, copy_stream);
            }
            if (e != cudaSuccess) { rc = cuda_fail(e, "cudaMemcpyAsync D2H"); break; }
        }
        if (rc == PIC_OK) {
            e = cudaStreamSynchronize(copy_stream);
            if (e != cudaSuccess) rc = cuda_fail(e, "cudaStreamSynchronize D2H");
        }
        mark("D2H done");
    } while (0);
    if (copy_stream) { cudaStreamSynchronize(copy_stream); cudaStreamDestroy(copy_stream); }
    if (sim) pic_destroy(sim);
    else cudaStreamSynchronize(stream);
    mark("sim destroyed");
    if (arena && !arena_cached) cudaFree(arena);
    if (arena_cached) { // kept for the next call
        std::lock_guard<std::mutex> lock(g_mem_mu);
        g_arena[arena_device].in_use = false;
    }
    mark("arena released");
    return rc;
}

// ------------------------------------------------------------------------------------------
// pic_deposit_static: the deposition for callers that may not allocate device memory (include/pic.h)
// ------------------------------------------------------------------------------------------
// The per-cell sums {sum (1-w), sum w} live in an array that is part of the library image instead of coming from the
// pool: 16 B * PIC_DEPOSIT_STATIC_MAX_NC = 16 MiB on every device that loads the library, for the life of the process.
// One array per device, shared by every call; it keeps the previous call's sums, which no call reads: entry c < nc is
// written by deposit_cell_kernel before deposit_node_kernel reads it, and entries >= nc are never read.
static __device__ __align__(256) double2 g_dep_static_cs[PIC_DEPOSIT_STATIC_MAX_NC];

// On the host, g_dep_static_cs is only the handle the runtime knows the array by, not an address a kernel can use.  Its
// device address differs per device and is looked up once per device (with that device current) by the first call.
static double2 *g_dep_static_addr[64] = {};
static std::mutex g_dep_static_mu;

static int dep_static_fail(int rc, const char *fmt, long long a = 0, long long b = 0)
{
    snprintf(g_err, sizeof g_err, fmt, a, b);
    return rc;
}

extern "C" int pic_deposit_static(const double *x_dev, const int32_t *offset_dev, int64_t n, int32_t nc, double dx,
                                  int32_t boundary, double weight, int accumulate, double *rho_dev, void *stream)
{
    // argument checks first: none of them touches CUDA
    if (!x_dev || !offset_dev || !rho_dev) return dep_static_fail(PIC_EINVAL, "pic_deposit_static: NULL device pointer");
    if (nc < 1) return dep_static_fail(PIC_EINVAL, "pic_deposit_static: nc = %lld, need nc >= 1", nc);
    if (nc > PIC_DEPOSIT_STATIC_MAX_NC)
        return dep_static_fail(PIC_ECAPACITY,
                               "pic_deposit_static: nc = %lld cells exceeds PIC_DEPOSIT_STATIC_MAX_NC = %lld, the size of the "
                               "built-in scratch array (use pic_deposit, or deposit the grid in pieces)",
                               nc, PIC_DEPOSIT_STATIC_MAX_NC);
    if (n < 0 || n >= (int64_t)INT_MAX - 64)
        return dep_static_fail(PIC_EINVAL, "pic_deposit_static: n = %lld outside [0, 2^31 - 64)", n);
    if (!std::isfinite(dx) || dx <= 0.0 || !std::isfinite(weight))
        return dep_static_fail(PIC_EINVAL, "pic_deposit_static: dx must be finite and positive, weight finite");
    if (boundary != PIC_PERIODIC && boundary != PIC_ABSORBING)
        return dep_static_fail(PIC_EINVAL, "pic_deposit_static: boundary = %lld is not a pic_boundary", boundary);

    int device = -1;
    CU(cudaGetDevice(&device));
    if (device < 0 || device >= 64) return dep_static_fail(PIC_EINVAL, "pic_deposit_static: device ordinal %lld not supported", device);
    double2 *cs = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_dep_static_mu);
        if (!g_dep_static_addr[device]) { // set-up, once per device: the first call on it (before any stream capture)
            void *p = nullptr;
            CU(cudaGetSymbolAddress(&p, g_dep_static_cs));
            g_dep_static_addr[device] = static_cast<double2 *>(p);
        }
        cs = g_dep_static_addr[device];
    }

    cudaStream_t st = static_cast<cudaStream_t>(stream);
    DepositArgs a{};
    a.x = x_dev;
    a.off = offset_dev;
    a.cs = cs;
    a.nc = nc;
    { volatile double inv = 1.0 / dx; a.inv_dx = inv; } // as boris_constants: one rounded division
    NvtxRange range("pic_deposit_static");
    const int lpc = n <= 448LL * nc ? 16 : 32; // the rule of deposit_enqueue, from n itself
    const long long threads = (long long)nc * lpc;
    const unsigned blocks = (unsigned)((threads + DEP_THREADS - 1) / DEP_THREADS);
    if (lpc == 16) deposit_cell_kernel<16><<<blocks, DEP_THREADS, 0, st>>>(a);
    else deposit_cell_kernel<32><<<blocks, DEP_THREADS, 0, st>>>(a);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "deposit_cell_kernel (static scratch)");
    deposit_node_kernel<<<(nc + 1 + 255) / 256, 256, 0, st>>>(cs, nc, boundary == PIC_PERIODIC ? 1 : 0, weight, accumulate ? 1 : 0, rho_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "deposit_node_kernel (static scratch)");
    return PIC_OK;
}
