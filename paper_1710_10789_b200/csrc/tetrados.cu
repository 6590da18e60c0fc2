// tetrados.cu -- C ABI (include/tetrados.h) and host planner of libtetrados.
//
// The planner owns: the per-block partial histograms, the fp64 merge buffer, host-mode staging
// buffers and a side stream.  Every step of the path runs in the kernels of tdos_kernels.cuh.
#include "../../include/tetrados.h"

#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "tdos_eigh.cuh"
#include "tdos_kernels.cuh"
#include "tdos_kweights.cuh"
#include "tdos_main5.cuh"

namespace {

thread_local char g_cuda_err[256] = "";

// cubes sampled by tdos_estimate when a plan chooses between its two main kernels per call
constexpr int kEstimateCubes = 2048;

// host mode: bytes of E + W per staged z-slab (copy/compute overlap granularity)
constexpr size_t kSlabBytes = (size_t)64 << 20;
// the first slabs are smaller (8 MB, doubling): the kernels start after 0.15 ms of copying instead of 1.2 ms
constexpr size_t kFirstSlabBytes = (size_t)8 << 20;

int cuda_fail(cudaError_t e, const char* what) {
    snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", what, cudaGetErrorString(e));
    cudaGetLastError();   // clear the sticky-less error state
    return TDOS_ECUDA;
}
#define CK(call)                                          \
    do {                                                  \
        cudaError_t e_ = (call);                          \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call); \
    } while (0)

// every entry point works on the plan's device and leaves the caller's current device as it found it
struct DeviceGuard {
    int prev = -1;
    cudaError_t err;
    explicit DeviceGuard(int dev) {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != dev) err = cudaSetDevice(dev);
        else if (err == cudaSuccess) prev = -1;   // nothing to restore
    }
    ~DeviceGuard() {
        if (prev >= 0) cudaSetDevice(prev);
    }
};
#define ON_DEVICE(dev)       \
    DeviceGuard guard_(dev); \
    if (guard_.err != cudaSuccess) return cuda_fail(guard_.err, "cudaSetDevice")

using tdos::MainParams;
typedef void (*main_kernel_t)(const MainParams);

struct Variant {
    main_kernel_t fn;      // tdos_main (generation 3) or tdos_main5 (generation 5)
    int MB, TX, TY, TZ, GL, NWARP;
    size_t smem;
    int gen = 3;                    // main kernel generation: 3 or 5
};

template <int TX, int TY, int TZ, int NWARP, int NORB>
Variant make_variant5() {
    Variant v{tdos::tdos_main5<TX, TY, TZ, NWARP, NORB>, 8, TX, TY, TZ, 2, NWARP,
              (size_t)NWARP * tdos::Cfg5<TX, TY, TZ>::bytes};
    v.gen = 5;
    return v;
}

// v5 configurations compiled in: the two tiles a default plan can pick (TDOS_TILE=<index> forces one); norb == 8 has
// its own instantiation with compile-time histogram offsets.  A build with -DTDOS_EXPERIMENTS adds the other shapes
// that were measured in DESIGN.md's experiments logs.
template <int NORB>
std::vector<Variant> variants5() {
    return {make_variant5<4, 4, 2, 16, NORB>(), make_variant5<2, 2, 8, 16, NORB>()
#ifdef TDOS_EXPERIMENTS
            , make_variant5<4, 2, 4, 16, NORB>(), make_variant5<4, 4, 2, 12, NORB>(), make_variant5<4, 4, 1, 16, NORB>()
#endif
    };
}

template <int MB, int TX, int TY, int TZ, int GL, int NWARP>
Variant make_variant() {
    return Variant{tdos::tdos_main<MB, TX, TY, TZ, GL, NWARP>, MB, TX, TY, TZ, GL, NWARP,
                   (size_t)NWARP * tdos::WarpCfg<MB, TX, TY, TZ>::bytes};
}

// fp64 accumulation (tdos_plan_set_accumulation): generation 3 with double-precision registers and partials; 12 warps
// leave room for the 64 accumulator registers of a block of 8 orbitals
template <int MB>
Variant make_variant64() {
    Variant v{tdos::tdos_main<MB, 4, 4, 2, 2, 12, true>, MB, 4, 4, 2, 2, 12, (size_t)12 * tdos::WarpCfg<MB, 4, 4, 2>::bytes};
    return v;
}
Variant variant64(int MB) {
    switch (MB) {
        case 1: return make_variant64<1>();
        case 2: return make_variant64<2>();
        case 4: return make_variant64<4>();
        default: return make_variant64<8>();
    }
}

// orbital-block width: the smallest of 1, 2, 4, 8 that holds norb (8 for norb > 8, several blocks)
int pick_mb(int norb) { return norb <= 1 ? 1 : norb <= 2 ? 2 : norb <= 4 ? 4 : 8; }

// Configurations compiled in: tile of cubes per warp, lanes per group, warps per block.  [0] is the kernel of plans
// that do not qualify for generation 5; blocks of 8 orbitals also have the two short-window kernels.
// TDOS_TILE=<index> forces one of them; -DTDOS_EXPERIMENTS adds the other shapes of the experiments logs.
template <int MB>
std::vector<Variant> variants_for() {
    std::vector<Variant> v = {make_variant<MB, 4, 4, 2, 2, 16>()};
    if constexpr (MB == 8) {
        // groups of ONE lane (chunks of 2 bins): the short-window kernel of plans that carry two
        v.push_back(make_variant<MB, 4, 4, 2, 1, 16>());
        v.push_back(make_variant<MB, 2, 2, 8, 1, 16>());
    }
#ifdef TDOS_EXPERIMENTS
    v.push_back(make_variant<MB, 4, 4, 2, 4, 16>());
    v.push_back(make_variant<MB, 4, 4, 4, 2, 12>());
    v.push_back(make_variant<MB, 4, 4, 4, 4, 12>());
    v.push_back(make_variant<MB, 4, 4, 2, 2, 20>());
#endif
    return v;
}
constexpr int kShortVariant = 1, kShortVariantZ8 = 2;   // indices into variants_for<8>()

std::vector<Variant> variants(int MB) {
    switch (MB) {
        case 1: return variants_for<1>();
        case 2: return variants_for<2>();
        case 4: return variants_for<4>();
        default: return variants_for<8>();
    }
}

}  // namespace

struct tdos_plan {
    int device = 0;
    int nk[3] = {0, 0, 0};
    int nb = 0, norb = 0, nE_max = 0;
    int num_sms = 0;
    size_t smem_optin = 0;        // cudaDevAttrMaxSharedMemoryPerBlockOptin
    Variant var{};                // the main kernel (generation 5 when the orbitals allow it, else 3)
    Variant var_short{};          // adaptive plans: generation 3, better when the windows are a few bins only
    // norb == 8 plans run tdos_main5<..., NORB = 8>, whose histogram layout is fixed at 8 rows; a selection of 9 rows
    // (8 orbitals + total, padded to 12) needs the same tile with a run-time row count
    Variant var_rows{};
    bool has_var_rows = false;
    int grid_rows = 0;
    bool adaptive = false;        // both kernels are enqueued; the device picks one per call (tdos_estimate)
    bool acc64 = false;           // tdos_plan_set_accumulation(TDOS_ACC_FP64): var64 runs, partials in fp64
    bool w64 = false;             // TDOS_ACC_FP64_ALL: var64 also evaluates the corner weights in fp64
    Variant var64{};
    int grid64 = 0;
    double* partial64 = nullptr;  // [grid64] rows [nE_max + 3][3 * norb_alloc], allocated when the mode is first set
    int blocks_per_sm = 0;
    int grid = 0;                 // blocks of `var`
    int grid_short = 0;           // blocks of `var_short`
    int nparts = 0;               // copies of the partial histogram = max(grid, grid_short)
    float* partial = nullptr;     // [nparts] rows [nE_max + 3][3 * norb]
    double* part64 = nullptr;     // [3][norb][nE_max]
    // [0..2] n_tb, n_eval, n_eval_mid of the last call; [3] work-item counter; [4..5] window sample (tdos_estimate)
    unsigned long long* counters = nullptr;
    cudaEvent_t done_ev = nullptr;   // end of the last call: the next call's stream waits for it (shared scratch)
    bool done_valid = false;
    // host-mode staging
    float* dE = nullptr;
    float* dW = nullptr;
    size_t dW_floats = 0;         // capacity of dW
    int cplx = 0;                 // the call in flight passes complex eigenvector elements instead of weights
    // the call in flight: rows the kernels work on (k_norb: output rows padded for the kernel in use), rows the caller
    // gets (k_nout), orbital selection (tetra_dos_select)
    int norb_alloc = 0;           // rows the scratch buffers hold: norb + 1 (selection + total), rounded up to 4
    int k_norb = 0, k_nout = 0;
    int sel_n = 0, sel_total = 0;
    short sel[32] = {};
    float* dOm = nullptr;
    float* dDos = nullptr;
    float* dNos = nullptr;
    cudaStream_t side = nullptr;
    cudaStream_t main = nullptr;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};   // [3] and [2] bracket the FMA probe
    // ring of event triples (before main kernel, after it, after merge+finalize), one per tetra_dos call
    static constexpr int kMaxSlabs = 32;
    cudaEvent_t cp_ev[kMaxSlabs] = {};   // host mode: slab s has arrived on the device
    static constexpr int kRing = 64;
    cudaEvent_t ring[kRing][3] = {};
    long long n_timed_calls = 0;   // tetra_dos (device path) calls since plan creation
    int cur_slot = 0;
    cudaStream_t last_stream = nullptr;
    bool last_stream_valid = false;
    bool timed = false;
    // the device-mode call being enqueued goes into a stream capture (CUDA graph): the plan's own events are left out
    // of it -- an event recorded inside a capture cannot be waited on or timed outside, and the other way round
    bool cap = false;
    long long last_items = 0, last_launches = 0;
};

// what a call without orbital selection works on
static void reset_call_state(tdos_plan* p) {
    p->cplx = 0;
    p->k_norb = p->k_nout = p->norb;
    p->sel_n = p->sel_total = 0;
}

extern "C" {

int tdos_version(void) { return 100; }

const char* tdos_strerror(int code) {
    switch (code) {
        case TDOS_OK: return "ok";
        case TDOS_EINVAL: return "invalid argument";
        case TDOS_ENOMEM: return "out of memory";
        case TDOS_ECUDA: return "CUDA error (see tdos_last_cuda_error)";
        case TDOS_EARCH: return "device is not compute capability 10.x (sm_100)";
        case TDOS_ESIZE: return "problem exceeds the built-in scratch of tetra_dos_static (norb * nE > TDOS_STATIC_MAX_CELLS)";
        default: return "unknown error code";
    }
}

const char* tdos_last_cuda_error(void) { return g_cuda_err; }

int tdos_plan_destroy(tdos_plan* p) {
    if (!p) return TDOS_OK;
    DeviceGuard guard_(p->device);
    if (p->side) cudaStreamSynchronize(p->side);
    if (p->main) cudaStreamSynchronize(p->main);
    cudaFree(p->partial);
    cudaFree(p->partial64);
    cudaFree(p->part64);
    cudaFree(p->counters);
    cudaFree(p->dE);
    cudaFree(p->dW);
    cudaFree(p->dOm);
    cudaFree(p->dDos);
    cudaFree(p->dNos);
    for (auto& e : p->ev)
        if (e) cudaEventDestroy(e);
    for (auto& e : p->cp_ev)
        if (e) cudaEventDestroy(e);
    if (p->done_ev) cudaEventDestroy(p->done_ev);
    for (auto& tr : p->ring)
        for (auto& e : tr)
            if (e) cudaEventDestroy(e);
    if (p->side) cudaStreamDestroy(p->side);
    if (p->main) cudaStreamDestroy(p->main);
    delete p;
    return TDOS_OK;
}

int tdos_plan_create(tdos_plan** out, int device, const int nk[3], int nb, int norb, int nE_max) {
    if (!out || !nk) return TDOS_EINVAL;
    if (nk[0] < 1 || nk[1] < 1 || nk[2] < 1 || nb < 1 || norb < 1 || nE_max < 1 || nE_max > TDOS_MAX_NE) return TDOS_EINVAL;
    if ((long long)nk[0] * nk[1] * nk[2] > 0x7fffffffLL) return TDOS_EINVAL;
    ON_DEVICE(device);
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, device));
    if (prop.major != 10) return TDOS_EARCH;

    tdos_plan* p = new (std::nothrow) tdos_plan;
    if (!p) return TDOS_ENOMEM;
    p->device = device;
    memcpy(p->nk, nk, sizeof(p->nk));
    p->nb = nb;
    p->norb = norb;
    p->norb_alloc = (norb + 1 + 3) & ~3;
    p->k_norb = p->k_nout = norb;
    p->nE_max = nE_max;
    p->num_sms = prop.multiProcessorCount;
    p->smem_optin = prop.sharedMemPerBlockOptin;

    const char* kv = getenv("TDOS_KERNEL");
    // generation 5 needs blocks of 8 orbitals to pay off; narrower problems use generation 3
    int gen = kv ? atoi(kv) : 5;
    if (gen == 5 && (norb < 5 || norb % 4 != 0)) gen = 3;   // tdos_main5: blocks of 8 orbitals, 16-byte vector reductions
    std::vector<Variant> vs = gen == 5 ? (norb == 8 ? variants5<8>() : variants5<0>()) : variants(pick_mb(norb));
    int sel = 0;
    // Tile shape of generation 5.  A tile whose bands span few energy bins keeps more (record, chunk) entries per
    // chunk.  The paper's workloads are layered materials sampled on grids like 60 x 60 x 10, with
    // the weak dispersion along z, so the default tile is long in z whenever the grid divides evenly (2 x 2 x 8
    // cubes, 15.1 ms on config 4 against 15.7 ms for 4 x 4 x 2); TDOS_TILE=<index> overrides it.
    if (gen == 5 && nk[2] % 8 == 0 && nk[0] % 2 == 0 && nk[1] % 2 == 0) sel = 1;
    if (const char* s = getenv("TDOS_TILE")) sel = atoi(s);
    if (sel < 0 || sel >= (int)vs.size()) sel = 0;
    p->var = vs[sel];

    // The shared-memory limit is an attribute of the kernel function, not of the plan: always the device maximum, so
    // that plans with different nE_max cannot lower each other's limit.
    auto setup = [&](const Variant& v, int* bps) -> cudaError_t {
        cudaError_t e = cudaFuncSetAttribute((const void*)v.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->smem_optin);
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(bps, (const void*)v.fn, v.NWARP * 32, v.smem);
        return e;
    };
    cudaError_t e = setup(p->var, &p->blocks_per_sm);
    if (e != cudaSuccess || p->blocks_per_sm < 1) {
        int rc = (e != cudaSuccess) ? cuda_fail(e, "kernel setup") : TDOS_ECUDA;
        delete p;
        return rc;
    }
#ifdef TDOS_EXPERIMENTS
    if (const char* s = getenv("TDOS_BLOCKS_PER_SM")) {   // fewer resident blocks, for occupancy experiments
        int b = atoi(s);
        if (b >= 1 && b < p->blocks_per_sm) p->blocks_per_sm = b;
    }
#endif
    p->grid = p->num_sms * p->blocks_per_sm;
    p->nparts = p->grid;
    if (gen == 5 && norb == 8) {
        p->var_rows = variants5<0>()[sel];
        int bps = 0;
        e = setup(p->var_rows, &bps);
        if (e != cudaSuccess || bps < 1) {
            int rc = (e != cudaSuccess) ? cuda_fail(e, "kernel setup") : TDOS_ECUDA;
            delete p;
            return rc;
        }
        if (bps > p->blocks_per_sm) bps = p->blocks_per_sm;
        p->has_var_rows = true;
        p->grid_rows = p->num_sms * bps;
    }
    // Without TDOS_KERNEL a plan on blocks of 8 orbitals carries both kernels: windows of a few bins only (config 5:
    // 3 bins on average) are served better by one record per tetrahedron (generation 3) than by three (generation 5).
    // Which one runs is decided per call on the device, from a sample of the windows (tdos_estimate).
    if (gen == 5 && !kv) {
        // one record per tetrahedron, chunks of 2 bins; long in z like the main kernel's tile when the grid divides
        p->var_short = variants(8)[(nk[2] % 8 == 0 && nk[0] % 2 == 0 && nk[1] % 2 == 0) ? kShortVariantZ8 : kShortVariant];
        int bps = 0;
        if (setup(p->var_short, &bps) == cudaSuccess && bps >= 1) {
            p->adaptive = true;
            p->grid_short = p->num_sms * bps;
            if (p->grid_short > p->nparts) p->nparts = p->grid_short;
        }
        cudaGetLastError();
    }

    const size_t hist = (size_t)3 * p->norb_alloc * ((size_t)nE_max + 3);
    if (cudaMalloc(&p->partial, hist * p->nparts * sizeof(float)) != cudaSuccess ||
        cudaMalloc(&p->part64, hist * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&p->counters, 8 * sizeof(unsigned long long)) != cudaSuccess) {
        cudaGetLastError();
        tdos_plan_destroy(p);
        return TDOS_ENOMEM;
    }
    if (cudaStreamCreateWithFlags(&p->side, cudaStreamNonBlocking) != cudaSuccess ||
        cudaStreamCreateWithFlags(&p->main, cudaStreamNonBlocking) != cudaSuccess) {
        int rc = cuda_fail(cudaGetLastError(), "cudaStreamCreate");
        tdos_plan_destroy(p);
        return rc;
    }
    if (cudaEventCreateWithFlags(&p->done_ev, cudaEventDisableTiming) != cudaSuccess) {
        int rc = cuda_fail(cudaGetLastError(), "cudaEventCreate");
        tdos_plan_destroy(p);
        return rc;
    }
    for (auto& ev : p->ev)
        if (cudaEventCreate(&ev) != cudaSuccess) {
            int rc = cuda_fail(cudaGetLastError(), "cudaEventCreate");
            tdos_plan_destroy(p);
            return rc;
        }
    for (auto& tr : p->ring)
        for (auto& ev : tr)
            if (cudaEventCreate(&ev) != cudaSuccess) {
                int rc = cuda_fail(cudaGetLastError(), "cudaEventCreate");
                tdos_plan_destroy(p);
                return rc;
            }
    *out = p;
    return TDOS_OK;
}

static int check_common(const tdos_plan* p, const float* E, const float* W, int layout, const float* omega, int nE) {
    if (!p || !E || !omega) return TDOS_EINVAL;
    if (nE < 1 || nE > p->nE_max || nE > TDOS_MAX_NE) return TDOS_EINVAL;
    if (layout != TDOS_AOS && layout != TDOS_SOA) return TDOS_EINVAL;
    if (!W && p->norb != 1) return TDOS_EINVAL;
    return TDOS_OK;
}

// rows of one block's partial histogram: generation 5 flushes whole chunks of 4 bins; both kernels use this layout
static int rows_per_block(int nE) { return (nE + 3) & ~3; }

// The plan's scratch (partials, counters, merge buffer) is shared by all calls: a call on another stream than the
// previous one waits for that one's end.
static int order_after_last_call(tdos_plan* p, cudaStream_t st) {
    if (p->cap) return TDOS_OK;   // a captured call is ordered by the graph's own dependencies (include/tetrados.h)
    if (p->done_valid && !(p->last_stream_valid && p->last_stream == st)) CK(cudaStreamWaitEvent(st, p->done_ev, 0));
    return TDOS_OK;
}
static int mark_end_of_call(tdos_plan* p, cudaStream_t st) {
    if (p->cap) return TDOS_OK;
    CK(cudaEventRecord(p->done_ev, st));
    p->done_valid = true;
    return TDOS_OK;
}
// is `st` being captured?  (sets p->cap for the helpers of this call)
static int note_capture(tdos_plan* p, cudaStream_t st) {
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    CK(cudaStreamIsCapturing(st, &cs));
    p->cap = (cs != cudaStreamCaptureStatusNone);
    return TDOS_OK;
}
// timing events of the ring: not recorded into a capture
static cudaError_t ring_record(tdos_plan* p, int which, cudaStream_t st) {
    return p->cap ? cudaSuccess : cudaEventRecord(p->ring[p->cur_slot][which], st);
}
// bookkeeping at the end of a device-mode call
static int end_of_device_call(tdos_plan* p, cudaStream_t st) {
    CK(ring_record(p, 2, st));
    if (!p->cap) {
        p->n_timed_calls++;
        p->timed = true;
    }
    const int rc = mark_end_of_call(p, st);
    p->cap = false;
    return rc;
}

// enqueue the main kernel for the cube slab [z_lo, z_hi); `first` also clears the block partials and the
// work counters (a call may cover the grid with several slab launches that accumulate into the same partials)
// `nz_arr` > 0: E and W hold only the nz_arr = z_hi - z_lo + 1 planes z_lo .. z_hi of the grid (the last one is the halo,
// plane z_hi mod N3), in that order (tetra_dos_partial_slab).  The kernels then run with base pointers moved back by z_lo
// planes and with N3 = z_hi + 1, so that no z index they form wraps and plane z lands on local plane z - z_lo.
static int enqueue_main(tdos_plan* p, const float* E, const float* W, int layout, const float* omega, int nE,
                        int z_lo, int z_hi, bool first, cudaStream_t st, int nz_arr = 0) {
    const long long nkt = (long long)p->nk[0] * p->nk[1] * (nz_arr > 0 ? nz_arr : p->nk[2]);
    MainParams mp{};
    mp.E = E;
    mp.W = W;
    mp.omega = omega;
    if (layout == TDOS_AOS) {
        mp.sEk = p->nb; mp.sEn = 1;
        mp.sWk = (long long)p->nb * p->norb; mp.sWn = p->norb; mp.sWm = 1;
    } else {
        mp.sEk = 1; mp.sEn = nkt;
        mp.sWk = 1; mp.sWn = (long long)p->norb * nkt; mp.sWm = nkt;
    }
    mp.N1 = p->nk[0]; mp.N2 = p->nk[1]; mp.N3 = p->nk[2];
    if (nz_arr > 0) {
        const long long k0 = (long long)p->nk[0] * p->nk[1] * z_lo;   // k-points in front of the slab
        const long long wfl = (W != nullptr && p->cplx) ? 2 : 1;      // floats per weight element
        mp.E = reinterpret_cast<const float*>(reinterpret_cast<uintptr_t>(E) - (uintptr_t)(k0 * mp.sEk) * sizeof(float));
        if (W) mp.W = reinterpret_cast<const float*>(reinterpret_cast<uintptr_t>(W) - (uintptr_t)(k0 * mp.sWk * wfl) * sizeof(float));
        mp.N3 = z_hi + 1;
    }
    mp.nb = p->nb; mp.norb = p->k_norb; mp.nE = nE;
    mp.nsel = p->sel_n; mp.total = p->sel_total; mp.norb_in = p->norb;
    memcpy(mp.sel, p->sel, sizeof(mp.sel));
    mp.nEp = rows_per_block(nE);
    mp.z_lo = z_lo; mp.z_hi = z_hi;
    mp.unitW = (W == nullptr);
    mp.cplx = (W != nullptr) ? p->cplx : 0;
    mp.partial = p->partial;
    mp.counters = p->counters;
    mp.next_item = reinterpret_cast<unsigned int*>(p->counters + 3);
    mp.partial64 = p->partial64;
    mp.w64 = (p->acc64 && p->w64) ? 1 : 0;
    const bool pair = p->adaptive && !p->acc64;   // both kernels enqueued, the device picks
    mp.est = pair ? p->counters + 4 : nullptr;

    const size_t hist = (size_t)3 * p->k_norb * mp.nEp;
    if (first) {
        if (p->acc64) CK(cudaMemsetAsync(p->partial64, 0, hist * p->grid64 * sizeof(double), st));
        else CK(cudaMemsetAsync(p->partial, 0, hist * p->nparts * sizeof(float), st));
        CK(cudaMemsetAsync(p->counters, 0, 8 * sizeof(unsigned long long), st));
        p->last_items = 0;
        p->last_launches = 0;
        if (pair && z_hi > z_lo) {   // sample the windows of this call's (first) slab: the device picks the kernel
            tdos::EstimateParams ep{};
            ep.E = mp.E; ep.omega = omega;
            ep.sEk = mp.sEk; ep.sEn = mp.sEn;
            ep.N1 = mp.N1; ep.N2 = mp.N2; ep.N3 = mp.N3; ep.nb = mp.nb; ep.nE = nE;
            ep.z_lo = z_lo; ep.z_hi = z_hi;
            const long long slab = (long long)mp.N1 * mp.N2 * (z_hi - z_lo);
            ep.n_cubes = (int)(slab < kEstimateCubes ? slab : kEstimateCubes);
            ep.est = p->counters + 4;
            const long long total = (long long)ep.n_cubes * 6 * mp.nb;
            tdos::tdos_estimate<<<(int)((total + 1023) / 1024), 256, 0, st>>>(ep);
            CK(cudaGetLastError());
            p->last_launches += 1;
        }
    } else {
        CK(cudaMemsetAsync(p->counters + 3, 0, sizeof(unsigned long long), st));
    }
    long long items_main = 0;
    for (int which = 0; which < (pair ? 2 : 1); ++which) {
        // more than 8 output rows on a norb == 8 plan: the generation-5 kernel with a run-time row count
        const bool rows = !which && p->has_var_rows && p->k_norb != 8;
        const Variant& v = p->acc64 ? p->var64 : which ? p->var_short : rows ? p->var_rows : p->var;
        const int vgrid = p->acc64 ? p->grid64 : which ? p->grid_short : rows ? p->grid_rows : p->grid;
        mp.ntx = (p->nk[0] + v.TX - 1) / v.TX;
        mp.nty = (p->nk[1] + v.TY - 1) / v.TY;
        mp.ntz = (z_hi - z_lo + v.TZ - 1) / v.TZ;
        mp.nmb = (p->k_norb + v.MB - 1) / v.MB;
        const long long items = (long long)mp.ntx * mp.nty * mp.ntz * p->nb * mp.nmb;
        if (items > 0x7fffffffLL) return TDOS_EINVAL;
        mp.n_items = (int)items;
        if (!which) items_main = items;
        // a block-wide copy of omega in shared memory if the device limit allows it
        size_t smem = v.smem;
        mp.om_smem = 0;
        if (v.smem + (size_t)nE * sizeof(float) <= p->smem_optin) {
            mp.om_smem = 1;
            smem += (size_t)nE * sizeof(float);
        }
        if (items > 0) {
            const long long blocks_needed = (items + v.NWARP - 1) / v.NWARP;
            const int grid = (int)((blocks_needed < vgrid) ? blocks_needed : vgrid);
            v.fn<<<grid, v.NWARP * 32, smem, st>>>(mp);
            CK(cudaGetLastError());
            p->last_launches += 1;
        }
    }
    p->last_items += items_main;
    p->last_stream = st;
    p->last_stream_valid = true;
    p->timed = false;
    return TDOS_OK;
}

// fp64 sum of the block partials -> part_out (device fp64 [3][norb][nE])
static int enqueue_merge(tdos_plan* p, int nE, double* part_out, cudaStream_t st) {
    const size_t hist = (size_t)3 * p->k_norb * nE;
    const int mblocks = (int)((hist + 255) / 256);
    if (p->acc64)
        tdos::tdos_merge64<<<mblocks, 256, 0, st>>>(p->partial64, p->grid64, p->k_norb, nE, rows_per_block(nE), part_out);
    else
        tdos::tdos_merge<<<mblocks, 256, 0, st>>>(p->partial, p->nparts, p->k_norb, nE, rows_per_block(nE), part_out);
    CK(cudaGetLastError());
    p->last_launches += 1;
    return TDOS_OK;
}

// zero partials, main kernel over [z_lo, z_hi), merge into part_out; events around the main kernel
static int enqueue_partial(tdos_plan* p, const float* E, const float* W, int layout, const float* omega, int nE,
                           int z_lo, int z_hi, double* part_out, cudaStream_t st, int nz_arr = 0) {
    int rc0 = note_capture(p, st);
    if (rc0) return rc0;
    rc0 = order_after_last_call(p, st);
    if (rc0) return rc0;
    CK(ring_record(p, 0, st));
    int rc = enqueue_main(p, E, W, layout, omega, nE, z_lo, z_hi, true, st, nz_arr);
    if (rc) return rc;
    CK(ring_record(p, 1, st));
    return enqueue_merge(p, nE, part_out, st);
}

static int enqueue_finalize(tdos_plan* p, const double* part, int nE, float* dos, float* nos, cudaStream_t st) {
    const double V = 1.0 / (24.0 * (double)p->nk[0] * (double)p->nk[1] * (double)p->nk[2]);
    tdos::tdos_finalize<<<p->k_nout, 1024, 0, st>>>(part, p->k_norb, nE, V, dos, nos);
    CK(cudaGetLastError());
    p->last_launches += 1;
    return TDOS_OK;
}

int tetra_dos_partial(tdos_plan* p, const float* E, const float* W, int layout, const float* omega, int nE,
                      int z_lo, int z_hi, double* part, void* cuda_stream) {
    int rc = check_common(p, E, W, layout, omega, nE);
    if (rc) return rc;
    if (!part || z_lo < 0 || z_hi > p->nk[2] || z_lo > z_hi) return TDOS_EINVAL;
    ON_DEVICE(p->device);
    reset_call_state(p);
    p->cur_slot = (int)(p->n_timed_calls % tdos_plan::kRing);
    rc = enqueue_partial(p, E, W, layout, omega, nE, z_lo, z_hi, part, (cudaStream_t)cuda_stream);
    if (rc) return rc;
    return end_of_device_call(p, (cudaStream_t)cuda_stream);
}

int tetra_dos_partial_slab(tdos_plan* p, const float* E, const float* W, int layout, const float* omega, int nE,
                           int z_lo, int z_hi, double* part, void* cuda_stream) {
    int rc = check_common(p, E, W, layout, omega, nE);
    if (rc) return rc;
    if (!part || z_lo < 0 || z_hi > p->nk[2] || z_lo >= z_hi) return TDOS_EINVAL;   // an empty slab has no arrays to pass
    ON_DEVICE(p->device);
    reset_call_state(p);
    p->cur_slot = (int)(p->n_timed_calls % tdos_plan::kRing);
    rc = enqueue_partial(p, E, W, layout, omega, nE, z_lo, z_hi, part, (cudaStream_t)cuda_stream, z_hi - z_lo + 1);
    if (rc) return rc;
    return end_of_device_call(p, (cudaStream_t)cuda_stream);
}

int tetra_dos_finalize(tdos_plan* p, const double* part, int nE, float* dos, float* nos, void* cuda_stream) {
    if (!p || !part || !dos || nE < 1 || nE > p->nE_max) return TDOS_EINVAL;
    ON_DEVICE(p->device);
    reset_call_state(p);
    return enqueue_finalize(p, part, nE, dos, nos, (cudaStream_t)cuda_stream);
}

static int run_device(tdos_plan* p, const float* E, const float* W, int layout, const float* omega, int nE,
                      float* dos, float* nos, cudaStream_t st) {
    p->cur_slot = (int)(p->n_timed_calls % tdos_plan::kRing);
    int rc = enqueue_partial(p, E, W, layout, omega, nE, 0, p->nk[2], p->part64, st);
    if (rc) return rc;
    rc = enqueue_finalize(p, p->part64, nE, dos, nos, st);
    if (rc) return rc;
    return end_of_device_call(p, st);
}

static int tetra_dos_impl(tdos_plan* p, const float* E, const float* W, int layout, const float* omega, int nE,
                          float* dos, float* nos, int memspace, void* cuda_stream);

int tetra_dos(tdos_plan* p, const float* E, const float* W, int layout, const float* omega, int nE, float* dos,
              float* nos, int memspace, void* cuda_stream) {
    if (p) reset_call_state(p);
    return tetra_dos_impl(p, E, W, layout, omega, nE, dos, nos, memspace, cuda_stream);
}

int tetra_dos_select(tdos_plan* p, const float* E, const float* W, int layout, const float* omega, int nE,
                     const int* orbitals, int nsel, int want_total, float* dos, float* nos, int memspace, void* cuda_stream) {
    if (!p || !W || nsel < 0 || nsel > 32 || (nsel > 0 && !orbitals) || (nsel == 0 && !want_total)) return TDOS_EINVAL;
    for (int j = 0; j < nsel; j++)
        if (orbitals[j] < 0 || orbitals[j] >= p->norb || orbitals[j] > 32767) return TDOS_EINVAL;   // kept in 16 bits
    reset_call_state(p);
    const int nout = nsel + (want_total ? 1 : 0);
    if (nout > p->norb + 1) return TDOS_EINVAL;   // the scratch buffers hold norb + 1 rows
    p->sel_n = nsel;
    p->sel_total = want_total ? 1 : 0;
    for (int j = 0; j < nsel; j++) p->sel[j] = (short)orbitals[j];
    p->k_nout = nout;
    // generation 5 works on whole blocks of 4 orbitals, at least 5 rows: the selection is padded with zero rows
    p->k_norb = (p->var.gen == 5 && !p->acc64) ? (nout <= 8 ? 8 : (nout + 3) & ~3) : nout;
    if (p->k_norb > p->norb_alloc) p->k_norb = p->norb_alloc;   // (norb_alloc = norb + 1 rounded up to 4 >= 8 for generation 5)
    const int rc = tetra_dos_impl(p, E, W, layout, omega, nE, dos, nos, memspace, cuda_stream);
    reset_call_state(p);
    return rc;
}

int tetra_dos_complex(tdos_plan* p, const float* E, const float* A, int layout, const float* omega, int nE,
                      float* dos, float* nos, int memspace, void* cuda_stream) {
    if (!p || !A) return TDOS_EINVAL;
    reset_call_state(p);
    p->cplx = 1;
    const int rc = tetra_dos_impl(p, E, A, layout, omega, nE, dos, nos, memspace, cuda_stream);
    p->cplx = 0;
    return rc;
}

static int tetra_dos_impl(tdos_plan* p, const float* E, const float* W, int layout, const float* omega, int nE,
                          float* dos, float* nos, int memspace, void* cuda_stream) {
    int rc = check_common(p, E, W, layout, omega, nE);
    if (rc) return rc;
    if (!dos) return TDOS_EINVAL;
    if (memspace != TDOS_DEVICE && memspace != TDOS_HOST) return TDOS_EINVAL;
    ON_DEVICE(p->device);
    if (memspace == TDOS_DEVICE) return run_device(p, E, W, layout, omega, nE, dos, nos, (cudaStream_t)cuda_stream);

    // ---- host mode: validate omega, stage in, run, stage out
    for (int i = 1; i < nE; i++)
        if (!(omega[i] > omega[i - 1])) return TDOS_EINVAL;
    const size_t nkt = (size_t)p->nk[0] * p->nk[1] * p->nk[2];
    const size_t nEb = (size_t)p->nE_max * sizeof(float);
    const size_t wfl = (size_t)(p->cplx ? 2 : 1);   // floats per orbital weight as the caller passes them
    if (p->dE && p->dW_floats < nkt * p->nb * p->norb * wfl) {   // a complex call after real ones: grow the staging buffer
        cudaFree(p->dW);
        p->dW = nullptr;
        p->dW_floats = 0;
        if (cudaMalloc(&p->dW, nkt * p->nb * p->norb * wfl * sizeof(float)) != cudaSuccess) {
            cudaGetLastError();
            cudaFree(p->dE); cudaFree(p->dOm); cudaFree(p->dDos); cudaFree(p->dNos);
            p->dE = p->dOm = p->dDos = p->dNos = nullptr;
            return TDOS_ENOMEM;
        }
        p->dW_floats = nkt * p->nb * p->norb * wfl;
    }
    if (!p->dE) {
        p->dW_floats = nkt * p->nb * p->norb * wfl;
        if (cudaMalloc(&p->dE, nkt * p->nb * sizeof(float)) != cudaSuccess ||
            cudaMalloc(&p->dW, p->dW_floats * sizeof(float)) != cudaSuccess ||
            cudaMalloc(&p->dOm, nEb) != cudaSuccess || cudaMalloc(&p->dDos, nEb * (p->norb + 1)) != cudaSuccess ||
            cudaMalloc(&p->dNos, nEb * (p->norb + 1)) != cudaSuccess) {
            cudaGetLastError();
            cudaFree(p->dE); cudaFree(p->dW); cudaFree(p->dOm); cudaFree(p->dDos); cudaFree(p->dNos);
            p->dE = p->dW = p->dOm = p->dDos = p->dNos = nullptr;
            p->dW_floats = 0;
            return TDOS_ENOMEM;
        }
    }
    // A0 ("called from a CPU code"): the grid is cut into z-slabs; slab s is copied on the
    // side stream while the main kernel works on slab s-1.  Copy s brings the planes (z_s, z_{s+1}] (copy 0
    // also plane 0), so the cubes of slab s -- which read planes z_s .. z_{s+1}, the last one wrapping to
    // plane 0 -- need copies 0..s only.
    cudaStream_t st = p->main, cp = p->side;
    p->cap = false;   // host mode runs on the plan's own streams, which are never captured
    rc = order_after_last_call(p, st);
    if (rc) return rc;
    const int N3 = p->nk[2];
    const size_t plane = (size_t)p->nk[0] * p->nk[1];
    const size_t total = nkt * p->nb * (1 + (W ? (size_t)p->norb * wfl : 0)) * sizeof(float);
    // slab boundaries zb[0..nslab]: 8, 16, 32 MB, then 64 MB each, then 32, 16, 8 MB -- a short first slab lets the
    // kernels start early (compute-bound case), a short last one leaves little to compute after the last copy
    // (copy-bound case)
    int zb[tdos_plan::kMaxSlabs + 1];
    int nslab = 0;
    {
        const double plane_bytes = (double)total / (double)N3;
        const double ramp = 7.0 * (double)kFirstSlabBytes;                     // 8 + 16 + 32 MB
        int nmid = (int)(((double)total - 2.0 * ramp) / (double)kSlabBytes + 0.999);
        if (nmid < 0) nmid = 0;
        if (nmid > tdos_plan::kMaxSlabs - 6) nmid = tdos_plan::kMaxSlabs - 6;
        const double covered = 2.0 * ramp + (double)nmid * (double)kSlabBytes;
        const double scale = (double)total > covered ? (double)total / covered : 1.0;
        double sizes[tdos_plan::kMaxSlabs];
        int ns = 0;
        for (int i = 0; i < 3; i++) sizes[ns++] = (double)(kFirstSlabBytes << i);
        for (int i = 0; i < nmid; i++) sizes[ns++] = (double)kSlabBytes;
        for (int i = 2; i >= 0; i--) sizes[ns++] = (double)(kFirstSlabBytes << i);
        zb[0] = 0;
        double acc = 0.0;
        // every slab is tiled from its own first plane, so a slab whose length is not a multiple of the tile's extent
        // in z ends in a layer of partly empty tiles: lengths are rounded to whole tiles (the short first slab, which
        // only has to start the kernels early, and the remainder at the end excepted)
        // (the largest tile extent among the kernels that may run this call; all are powers of two)
        int tz = p->acc64 ? p->var64.TZ : p->var.TZ;
        if (!p->acc64 && p->adaptive && p->var_short.TZ > tz) tz = p->var_short.TZ;
        for (int i = 0; i < ns && zb[nslab] < N3; i++) {
            acc += sizes[i] * scale;
            int z = (int)(acc / plane_bytes + 0.5);
            if (z <= zb[nslab]) z = zb[nslab] + 1;
            if (i > 0 && tz > 1) {
                int len = ((z - zb[nslab] + tz / 2) / tz) * tz;
                if (len < tz) len = tz;
                z = zb[nslab] + len;
            }
            if (z > N3 || i == ns - 1) z = N3;
            zb[++nslab] = z;
        }
        if (zb[nslab] < N3) zb[nslab] = N3;
    }
    for (int i = 0; i < nslab; i++)
        if (!p->cp_ev[i]) CK(cudaEventCreateWithFlags(&p->cp_ev[i], cudaEventDisableTiming));
    CK(cudaMemcpyAsync(p->dOm, omega, (size_t)nE * sizeof(float), cudaMemcpyHostToDevice, st));
    p->cur_slot = (int)(p->n_timed_calls % tdos_plan::kRing);
    CK(cudaEventRecord(p->ring[p->cur_slot][0], st));
    for (int sidx = 0; sidx < nslab; sidx++) {
        const int z_lo = zb[sidx], z_hi = zb[sidx + 1];
        const int c_lo = sidx == 0 ? 0 : z_lo + 1, c_hi = (z_hi + 1 < N3) ? z_hi + 1 : N3;
        if (c_hi > c_lo) {
            const size_t k0 = (size_t)c_lo * plane, nk_s = (size_t)(c_hi - c_lo) * plane;
            if (layout == TDOS_AOS) {
                const size_t se = (size_t)p->nb, sw = (size_t)p->nb * p->norb * wfl;
                CK(cudaMemcpyAsync(p->dE + k0 * se, E + k0 * se, nk_s * se * sizeof(float), cudaMemcpyHostToDevice, cp));
                if (W)
                    CK(cudaMemcpyAsync(p->dW + k0 * sw, W + k0 * sw, nk_s * sw * sizeof(float), cudaMemcpyHostToDevice, cp));
            } else {   // SoA: one strided copy of the slab's k-range for every band (and orbital)
                const size_t pitch = nkt * sizeof(float);
                CK(cudaMemcpy2DAsync(p->dE + k0, pitch, E + k0, pitch, nk_s * sizeof(float), (size_t)p->nb,
                                     cudaMemcpyHostToDevice, cp));
                if (W)
                    CK(cudaMemcpy2DAsync(p->dW + k0 * wfl, pitch * wfl, W + k0 * wfl, pitch * wfl, nk_s * wfl * sizeof(float),
                                         (size_t)p->nb * p->norb, cudaMemcpyHostToDevice, cp));
            }
        }
        CK(cudaEventRecord(p->cp_ev[sidx], cp));
        CK(cudaStreamWaitEvent(st, p->cp_ev[sidx], 0));
        rc = enqueue_main(p, p->dE, W ? p->dW : nullptr, layout, p->dOm, nE, z_lo, z_hi, sidx == 0, st);
        if (rc) return rc;
    }
    CK(cudaEventRecord(p->ring[p->cur_slot][1], st));
    rc = enqueue_merge(p, nE, p->part64, st);
    if (rc) return rc;
    rc = enqueue_finalize(p, p->part64, nE, p->dDos, p->dNos, st);
    if (rc) return rc;
    CK(cudaEventRecord(p->ring[p->cur_slot][2], st));
    p->n_timed_calls++;
    p->timed = true;
    CK(cudaMemcpyAsync(dos, p->dDos, (size_t)p->k_nout * nE * sizeof(float), cudaMemcpyDeviceToHost, st));
    if (nos) CK(cudaMemcpyAsync(nos, p->dNos, (size_t)p->k_nout * nE * sizeof(float), cudaMemcpyDeviceToHost, st));
    rc = mark_end_of_call(p, st);
    if (rc) return rc;
    CK(cudaStreamSynchronize(st));
    return TDOS_OK;
}

int tetra_weights(tdos_plan* p, const float* E, int layout, const float* energies, int nW, float* wk, float* dwk,
                  void* cuda_stream) {
    if (!p || !E || !energies || !wk || nW < 1) return TDOS_EINVAL;
    if (layout != TDOS_AOS && layout != TDOS_SOA) return TDOS_EINVAL;
    ON_DEVICE(p->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long long nkt = (long long)p->nk[0] * p->nk[1] * p->nk[2];
    tdos::KWeightParams kp{};
    kp.E = E;
    kp.energies = energies;
    if (layout == TDOS_AOS) { kp.sEk = p->nb; kp.sEn = 1; } else { kp.sEk = 1; kp.sEn = nkt; }
    kp.N1 = p->nk[0]; kp.N2 = p->nk[1]; kp.N3 = p->nk[2];
    kp.nb = p->nb; kp.nW = nW;
    kp.V = (float)(1.0 / (24.0 * (double)nkt));
    kp.wk = wk;
    kp.dwk = dwk;
    const size_t bytes = (size_t)nW * p->nb * nkt * sizeof(float);
    CK(cudaMemsetAsync(wk, 0, bytes, st));
    if (dwk) CK(cudaMemsetAsync(dwk, 0, bytes, st));
    const long long total = nkt * 6 * p->nb;
    long long blocks = (total + 255) / 256;
    if (blocks > (long long)p->num_sms * 32) blocks = (long long)p->num_sms * 32;
    tdos::tdos_kweights<<<(int)blocks, 256, 0, st>>>(kp);
    CK(cudaGetLastError());
    return TDOS_OK;
}

int tetra_eigh(tdos_plan* p, const float* H, float* E, float* A, void* cuda_stream) {
    if (!p || !H || !E || !A) return TDOS_EINVAL;
    if (p->nb != p->norb || p->nb > 16) return TDOS_EINVAL;   // square problems of order <= 16
    ON_DEVICE(p->device);
    tdos::EighParams ep{};
    ep.H = reinterpret_cast<const float2*>(H);
    ep.E = E;
    ep.A = reinterpret_cast<float2*>(A);
    ep.nmat = (long long)p->nk[0] * p->nk[1] * p->nk[2];
    ep.nb = p->nb;
    if (p->nb <= 8) {        // 8 lanes per matrix
        ep.sweeps = 10;
        const long long threads = ep.nmat * 8;
        tdos::tdos_eigh8<<<(unsigned)((threads + 127) / 128), 128, 0, (cudaStream_t)cuda_stream>>>(ep);
    } else {                 // orders 9..16: 16 lanes per matrix
        ep.sweeps = 14;
        const long long threads = ep.nmat * 16;
        tdos::tdos_eigh_n<16><<<(unsigned)((threads + 127) / 128), 128, 0, (cudaStream_t)cuda_stream>>>(ep);
    }
    CK(cudaGetLastError());
    return TDOS_OK;
}

int tetra_dos_simple(const float* E, const float* W, int Nk, int nb, int norb, float omega_min, float omega_max,
                     int nE, float* dos, float* nos) {
    if (!E || !dos || Nk < 1 || nE < 1 || nE > TDOS_MAX_NE) return TDOS_EINVAL;
    if (nE > 1 && !(omega_max > omega_min)) return TDOS_EINVAL;
    int dev = 0;
    CK(cudaGetDevice(&dev));
    std::vector<float> om;
    try {
        om.resize(nE);
    } catch (...) {
        return TDOS_ENOMEM;
    }
    for (int i = 0; i < nE; i++)
        om[i] = (nE == 1) ? omega_min
                          : (float)((double)omega_min + (double)i * (((double)omega_max - (double)omega_min) / (double)(nE - 1)));
    const int nk[3] = {Nk, Nk, Nk};
    tdos_plan* p = nullptr;
    int rc = tdos_plan_create(&p, dev, nk, nb, norb, nE);
    if (rc) return rc;
    rc = tetra_dos(p, E, W, TDOS_AOS, om.data(), nE, dos, nos, TDOS_HOST, nullptr);
    tdos_plan_destroy(p);
    return rc;
}

int tdos_plan_set_accumulation(tdos_plan* p, int mode) {
    if (!p || (mode != TDOS_ACC_FP32 && mode != TDOS_ACC_FP64 && mode != TDOS_ACC_FP64_ALL)) return TDOS_EINVAL;
    ON_DEVICE(p->device);
    if (mode != TDOS_ACC_FP32 && !p->partial64) {
        p->var64 = variant64(pick_mb(p->norb));
        int bps = 0;
        cudaError_t e = cudaFuncSetAttribute((const void*)p->var64.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->smem_optin);
        if (e == cudaSuccess)
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, (const void*)p->var64.fn, p->var64.NWARP * 32, p->var64.smem);
        if (e != cudaSuccess || bps < 1) return (e != cudaSuccess) ? cuda_fail(e, "kernel setup") : TDOS_ECUDA;
        p->grid64 = p->num_sms * bps;
        const size_t hist = (size_t)3 * p->norb_alloc * ((size_t)p->nE_max + 3);
        if (cudaMalloc(&p->partial64, hist * p->grid64 * sizeof(double)) != cudaSuccess) {
            cudaGetLastError();
            p->partial64 = nullptr;
            return TDOS_ENOMEM;
        }
    }
    if (p->last_stream_valid) CK(cudaStreamSynchronize(p->last_stream));   // no call in flight changes its kernels
    p->acc64 = (mode != TDOS_ACC_FP32);
    p->w64 = (mode == TDOS_ACC_FP64_ALL);
    return TDOS_OK;
}

int tdos_plan_info(const tdos_plan* p, long long what[8]) {
    if (!p || !what) return TDOS_EINVAL;
    what[0] = p->grid;
    what[1] = p->var.NWARP * 32;
    what[2] = (long long)p->var.smem;
    what[3] = p->last_items;
    what[4] = p->last_launches;
    what[5] = p->var.TX;
    what[6] = p->var.TY;
    what[7] = p->var.TZ;
    return TDOS_OK;
}

int tdos_last_counters(tdos_plan* p, long long cnt[4]) {
    if (!p || !cnt || !p->last_stream_valid) return TDOS_EINVAL;
    ON_DEVICE(p->device);
    CK(cudaStreamSynchronize(p->last_stream));
    unsigned long long h[6];
    CK(cudaMemcpy(h, p->counters, sizeof(h), cudaMemcpyDeviceToHost));
    const int gen = p->acc64 ? 3 : p->adaptive ? tdos::wanted_generation(h[4], h[5]) : p->var.gen;   // what the device decided
    cnt[0] = (long long)h[0];
    cnt[1] = (long long)h[1];
    cnt[2] = gen == 5 ? (long long)h[2] : -1;
    cnt[3] = gen;
    return TDOS_OK;
}

int tdos_kernel_ms(tdos_plan* p, int ncalls, float* main_ms, float* merge_ms) {
    if (!p || !main_ms || !merge_ms || !p->timed || ncalls < 1 || ncalls > tdos_plan::kRing ||
        ncalls > p->n_timed_calls)
        return TDOS_EINVAL;
    ON_DEVICE(p->device);
    double a = 0.0, b = 0.0;
    for (int j = 0; j < ncalls; j++) {
        cudaEvent_t* tr = p->ring[(p->n_timed_calls - 1 - j) % tdos_plan::kRing];
        CK(cudaEventSynchronize(tr[2]));
        float x = 0.f, y = 0.f;
        CK(cudaEventElapsedTime(&x, tr[0], tr[1]));
        CK(cudaEventElapsedTime(&y, tr[1], tr[2]));
        a += x;
        b += y;
    }
    *main_ms = (float)(a / ncalls);
    *merge_ms = (float)(b / ncalls);
    return TDOS_OK;
}

int tdos_last_kernel_ms(tdos_plan* p, float* main_ms, float* merge_ms) { return tdos_kernel_ms(p, 1, main_ms, merge_ms); }

int tdos_fp32_fma_probe(tdos_plan* p, int packed, double* tflops) {
    if (!p || !tflops) return TDOS_EINVAL;
    ON_DEVICE(p->device);
    const int iters = 4096, blocks = p->num_sms * 8, threads = 256;
    float* d = nullptr;
    CK(cudaMalloc(&d, sizeof(float)));
    cudaStream_t st = p->main;
    float best = 1e30f;
    for (int rep = 0; rep < 5; rep++) {
        CK(cudaEventRecord(p->ev[3], st));
        if (packed)
            tdos::tdos_fma_probe<true><<<blocks, threads, 0, st>>>(d, iters, 1.0001f, 1e-7f);
        else
            tdos::tdos_fma_probe<false><<<blocks, threads, 0, st>>>(d, iters, 1.0001f, 1e-7f);
        CK(cudaGetLastError());
        CK(cudaEventRecord(p->ev[2], st));
        CK(cudaEventSynchronize(p->ev[2]));
        float ms = 0;
        CK(cudaEventElapsedTime(&ms, p->ev[3], p->ev[2]));
        if (rep > 0 && ms < best) best = ms;
    }
    p->timed = false;
    cudaFree(d);
    const double fmas = (double)blocks * threads * iters * 16.0;
    *tflops = 2.0 * fmas / (best * 1e-3) / 1e12;
    return TDOS_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// tetra_dos_static: the path for callers that must not allocate (include/tetrados.h).  All scratch of one call sits in
// this array, which is part of the library image: the driver places a copy on every GPU that loads the library and
// keeps it until the process ends.  Layout (bytes):
//     [0, 64)                          work counters of tdos_main (8 x u64)
//     [256, 256 + 3*MAX_CELLS*8)       fp64 merge buffer  part[3][norb][nE]
//     [.., .. + 16 MiB)                block-partial histograms, as many copies of [nEp][3*norb] floats as fit
// NOTE for maintainers: in HOST code the name g_static_scratch is only a handle for the runtime's symbol table, not
// a device address.  Passing it (or &g_static_scratch[0]) to a kernel would hand the GPU a host-side address.  Host
// code gets the real address from cudaGetSymbolAddress, once per device, in static_setup() below.
namespace {

constexpr size_t kStaticCountersOff = 0;
constexpr size_t kStaticMergeOff = 256;
constexpr size_t kStaticMergeBytes = (size_t)3 * TDOS_STATIC_MAX_CELLS * sizeof(double);
constexpr size_t kStaticPartialOff = kStaticMergeOff + kStaticMergeBytes;
constexpr size_t kStaticPartialBytes = (size_t)16 << 20;
static_assert(kStaticPartialOff % 256 == 0, "partials start on a 256-byte boundary");
static_assert(kStaticPartialOff + kStaticPartialBytes == (size_t)TDOS_STATIC_SCRATCH_BYTES, "header and layout agree");

static __device__ __align__(256) unsigned char g_static_scratch[TDOS_STATIC_SCRATCH_BYTES];

// what the first call on a device finds out and later calls reuse
struct StaticDevice {
    bool ready = false;
    unsigned char* scratch = nullptr;   // device address of g_static_scratch on this device
    int num_sms = 0;
    size_t smem_optin = 0;
    Variant var[4];                     // tdos_main for orbital blocks of 1, 2, 4, 8
    int blocks_per_sm[4] = {0, 0, 0, 0};
};
constexpr int kStaticMaxDevices = 64;
StaticDevice g_static_dev[kStaticMaxDevices];
std::mutex g_static_mutex;

int mb_index(int MB) { return MB == 1 ? 0 : MB == 2 ? 1 : MB == 4 ? 2 : 3; }

// Runs with `dev` current.  Nothing here allocates: symbol lookup, attribute queries, a function attribute.
int static_setup(int dev, StaticDevice** out) {
    if (dev < 0 || dev >= kStaticMaxDevices) return TDOS_EINVAL;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticDevice& sd = g_static_dev[dev];
    if (!sd.ready) {
        int major = 0, sms = 0, optin = 0;
        CK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
        if (major != 10) return TDOS_EARCH;
        CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        CK(cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
        void* addr = nullptr;
        CK(cudaGetSymbolAddress(&addr, g_static_scratch));
        if (!addr) return TDOS_ECUDA;
        const int mbs[4] = {1, 2, 4, 8};
        for (int i = 0; i < 4; i++) {
            sd.var[i] = variants(mbs[i])[0];   // 4 x 4 x 2 cubes per warp, groups of 2 lanes, 16 warps
            CK(cudaFuncSetAttribute((const void*)sd.var[i].fn, cudaFuncAttributeMaxDynamicSharedMemorySize, optin));
            CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&sd.blocks_per_sm[i], (const void*)sd.var[i].fn,
                                                             sd.var[i].NWARP * 32, sd.var[i].smem));
            if (sd.blocks_per_sm[i] < 1) return TDOS_ECUDA;
        }
        sd.scratch = static_cast<unsigned char*>(addr);
        sd.num_sms = sms;
        sd.smem_optin = (size_t)optin;
        sd.ready = true;
    }
    *out = &sd;
    return TDOS_OK;
}

}  // namespace

extern "C" int tetra_dos_static(const int nk[3], int nb, int norb, const float* E, const float* W, int layout,
                                const float* omega, int nE, float* dos, float* nos, void* cuda_stream) {
    if (!nk || !E || !omega || !dos) return TDOS_EINVAL;
    if (nk[0] < 1 || nk[1] < 1 || nk[2] < 1 || nb < 1 || norb < 1 || nE < 1 || nE > TDOS_MAX_NE) return TDOS_EINVAL;
    if (layout != TDOS_AOS && layout != TDOS_SOA) return TDOS_EINVAL;
    if (!W && norb != 1) return TDOS_EINVAL;
    const long long nkt = (long long)nk[0] * nk[1] * nk[2];
    if (nkt > 0x7fffffffLL) return TDOS_EINVAL;
    const int nEp = rows_per_block(nE);
    if ((long long)norb * nEp > TDOS_STATIC_MAX_CELLS) return TDOS_ESIZE;   // before anything touches the device

    int dev = 0;
    CK(cudaGetDevice(&dev));
    StaticDevice* sd = nullptr;
    int rc = static_setup(dev, &sd);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;

    unsigned long long* counters = reinterpret_cast<unsigned long long*>(sd->scratch + kStaticCountersOff);
    double* merged = reinterpret_cast<double*>(sd->scratch + kStaticMergeOff);
    float* partial = reinterpret_cast<float*>(sd->scratch + kStaticPartialOff);

    const int mi = mb_index(pick_mb(norb));
    const Variant& v = sd->var[mi];
    MainParams mp{};
    mp.E = E;
    mp.W = W;
    mp.omega = omega;
    if (layout == TDOS_AOS) {
        mp.sEk = nb; mp.sEn = 1;
        mp.sWk = (long long)nb * norb; mp.sWn = norb; mp.sWm = 1;
    } else {
        mp.sEk = 1; mp.sEn = nkt;
        mp.sWk = 1; mp.sWn = (long long)norb * nkt; mp.sWm = nkt;
    }
    mp.N1 = nk[0]; mp.N2 = nk[1]; mp.N3 = nk[2];
    mp.nb = nb; mp.norb = norb; mp.nE = nE;
    mp.norb_in = norb;
    mp.nEp = nEp;
    mp.z_lo = 0; mp.z_hi = nk[2];
    mp.unitW = (W == nullptr);
    mp.ntx = (nk[0] + v.TX - 1) / v.TX;
    mp.nty = (nk[1] + v.TY - 1) / v.TY;
    mp.ntz = (nk[2] + v.TZ - 1) / v.TZ;
    mp.nmb = (norb + v.MB - 1) / v.MB;
    const long long items = (long long)mp.ntx * mp.nty * mp.ntz * nb * mp.nmb;
    if (items > 0x7fffffffLL) return TDOS_EINVAL;
    mp.n_items = (int)items;
    mp.est = nullptr;   // this kernel runs unconditionally
    mp.partial = partial;
    mp.partial64 = nullptr;
    mp.counters = counters;
    mp.next_item = reinterpret_cast<unsigned int*>(counters + 3);

    // one private histogram per block: as many blocks as histograms fit into the buffer, at most what the GPU holds
    // and what the work needs (the size check above guarantees at least 42)
    const size_t hist = (size_t)3 * norb * nEp;
    long long grid = (long long)(kStaticPartialBytes / (hist * sizeof(float)));
    const long long resident = (long long)sd->num_sms * sd->blocks_per_sm[mi];
    const long long blocks_needed = (items + v.NWARP - 1) / v.NWARP;
    if (grid > resident) grid = resident;
    if (grid > blocks_needed) grid = blocks_needed;
    if (grid < 1) grid = 1;

    size_t smem = v.smem;
    if (v.smem + (size_t)nE * sizeof(float) <= sd->smem_optin) {   // block-wide copy of omega in shared memory
        mp.om_smem = 1;
        smem += (size_t)nE * sizeof(float);
    }

    // the buffer still holds the previous call's sums: clear exactly what this call reads back
    CK(cudaMemsetAsync(partial, 0, hist * (size_t)grid * sizeof(float), st));
    CK(cudaMemsetAsync(counters, 0, 8 * sizeof(unsigned long long), st));
    v.fn<<<(int)grid, v.NWARP * 32, smem, st>>>(mp);
    CK(cudaGetLastError());
    // the merge writes every element of part[3][norb][nE] that finalize reads: no clearing needed
    const size_t cells = (size_t)3 * norb * nE;
    tdos::tdos_merge<<<(int)((cells + 255) / 256), 256, 0, st>>>(partial, (int)grid, norb, nE, nEp, merged);
    CK(cudaGetLastError());
    const double V = 1.0 / (24.0 * (double)nk[0] * (double)nk[1] * (double)nk[2]);
    tdos::tdos_finalize<<<norb, 1024, 0, st>>>(merged, norb, nE, V, dos, nos);
    CK(cudaGetLastError());
    return TDOS_OK;
}
