// gf_api.cu -- the C ABI of include/gf.h: argument checks, the context, the host-side fix loop
// and the mixed-precision hand-off.  No arithmetic of the method runs on the
// host: every step is one of the kernels in gf_sweep.cu / gf_aux.cu, the reductions included
// (sums over time slices and the normalisations of F and theta are done by reduce_slices_kernel);
// the host compares theta with the target and, in Coulomb gauge, takes the maximum over slices.
#include <cuda.h>

#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

#include "../../include/gf.h"
#include "gf_internal.h"

using namespace gf;

extern "C" int gf_transform_identity(gf_ctx* ctx, int precision);
static int write_identity(gf_ctx* ctx, int precision);
extern "C" int gf_coulomb_finish(gf_ctx* ctx, int precision);
static int upload_mask(gf_ctx* ctx);
static int sync_and_check(gf_ctx* ctx, const char* what);

namespace {
constexpr int kMeasureBlock = 128;
constexpr int kMaxNt = 4096;
constexpr int kAsyncSlots = 16;
constexpr int kRunAhead = 8;          // most evaluation blocks the fix loop keeps enqueued ahead of the one it reads
}

struct gf_ctx {
    int dims[4];
    int gauge, recon;
    void* links[2];             // [PREC_F32], [PREC_F64]
    void* gtrans[2];            // accumulated transformation per precision (gf_set_transform), or NULL
    int defer_temporal;         // Coulomb: sweeps record G(x) and leave the temporal links to gf_coulomb_finish
    int freeze_slices;          // Coulomb: gf_fix_until stops sweeping slices whose theta_t is below the target
    int pending[2];             // deferred temporal update outstanding for the field of that precision
    uint16_t* dev_list;         // workspace: the time slices still being swept (ascending)
    uint16_t* host_list;        // pinned staging copy of it
    uint8_t* host_mask;         // one byte per time slice, 0 = frozen: what the list is built from
    int n_active;               // entries of the list
    int mask_on;                // the sweeps cover the listed slices only
    double handoff;             // mixed precision: theta at which the fp32 phase hands over to fp64
    double stall;               // mixed precision: the fp32 phase also ends when theta > stall * previous theta (0 = off)
    // slab decomposition along t (gf_set_slab): this context holds N_t local slices of a lattice nranks times as long
    int slab_rank, slab_n;
    void* prev_links[2];        // field of the slab below (per precision); NULL = own (one slab)
    void* next_links[2];        // field of the slab above
    uint32_t *flag_own, *flag_prev, *flag_next;   // device words: number of operations completed by that slab
    uint32_t epoch;             // operations this slab has enqueued
    CUresult (*wait32)(CUstream, CUdeviceptr, cuuint32_t, unsigned int);
    CUresult (*write32)(CUstream, CUdeviceptr, cuuint32_t, unsigned int);
    int device;                 // CUDA device the buffers and the stream belong to; every entry point runs under it
    double* workspace;
    double* partials;           // workspace: per-block partial sums
    double* slice_tmp;          // workspace: 2 doubles per time slice (reduce_slices_kernel, whole-lattice sums)
    uint32_t* reduce_counter;   // workspace: blocks of the last reduction stage that have finished (zero between launches)
    uint32_t* stop_dev;         // workspace: zero except while a run-ahead fix loop has reached its target on the device
    int reunit_every;           // gf_fix_until re-projects the swept field onto SU(3) every so many iterations (0 = never)
    int runahead;               // evaluation blocks gf_fix_until keeps in flight (0 = wait for every theta before going on)
    cudaEvent_t fix_events[8];  // one per block in flight
    double* slice_out;          // 2 doubles per time slice, written by the last reduction kernel: the DEVICE ADDRESS OF
                                // host_pinned (zero-copy: the result is in host memory when the stream has drained)
    double* host_pinned;        // 2 * Nt doubles
    double* host_slots;         // (kAsyncSlots + kRunAhead) x 2 * Nt doubles (pinned): results of gf_measure_async, then
                                // the ring the run-ahead fix loop reads its evaluations from
    double* slots_dev;          // device address of host_slots
    int slot_precision[16];     // precision measured into the slot, or -1 when empty
    cudaStream_t stream;
    uint64_t seed;
    uint32_t counter;
    Geom G;
    MeasureGrid mg;
    size_t V;
    int lanes[2], block[2];
    int zigzag;                 // alternate the traversal direction of consecutive half-sweeps
    uint64_t sweeps;            // half-sweeps enqueued so far (selects the direction)
    int solver_mode;            // fp32 storage: K and the SU(2) solves in GF_F32, GF_F64 or GF_SOLVER_AUTO
    uint64_t launches;
    char err[256];
};

static int fail(gf_ctx* ctx, int code, const char* fmt, ...)
{
    if (ctx) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(ctx->err, sizeof(ctx->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

static int cuda_fail(gf_ctx* ctx, cudaError_t e, const char* what)
{
    return fail(ctx, GF_ECUDA, "%s: %s", what, cudaGetErrorString(e));
}

// Makes the context's device current for the duration of a call (streams, launches and stream memory
// operations need it) and restores the caller's device afterwards: one process may drive contexts on
// several GPUs (slabs.SlabSet).
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const gf_ctx* ctx)
    {
        if (ctx && cudaGetDevice(&prev) == cudaSuccess && prev != ctx->device) switched = cudaSetDevice(ctx->device) == cudaSuccess;
    }
    ~DeviceGuard()
    {
        if (switched) cudaSetDevice(prev);
    }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;
};

static bool dims_ok(const int dims[4])
{
    if (!dims) return false;
    uint64_t V = 1;
    for (int i = 0; i < 4; ++i) {
        if (dims[i] < 2 || (dims[i] & 1)) return false;
        V *= (uint64_t)dims[i];
    }
    return dims[0] <= kMaxNt && V < (uint64_t(1) << 32);
}

static MeasureGrid measure_grid(const int dims[4])
{
    MeasureGrid mg;
    mg.Sh = (uint32_t)((uint64_t)dims[1] * dims[2] * dims[3] / 2);
    mg.block = kMeasureBlock;
    mg.bpp = (mg.Sh + mg.block - 1) / mg.block;
    mg.slice_list = nullptr;
    mg.n_listed = 0;
    return mg;
}

extern "C" size_t gf_storage_bytes(const int dims[4], int precision, int recon)
{
    if (!dims_ok(dims) || (precision != GF_F32 && precision != GF_F64) || (recon != 18 && recon != 12)) return 0;
    const size_t Vh = (size_t)dims[0] * dims[1] * dims[2] * dims[3] / 2;
    const size_t tile = precision == GF_F64 ? Tile<double>::W : Tile<float>::W;     // sites per layout tile (gf_device.cuh)
    return (Vh + tile - 1) / tile * tile * 8 * (size_t)recon * (precision == GF_F64 ? 8 : 4);
}

extern "C" size_t gf_transform_bytes(const int dims[4], int precision, int recon)
{
    return gf_storage_bytes(dims, precision, recon) / 4;      // one matrix per site, links have four
}

extern "C" size_t gf_workspace_bytes(const int dims[4])
{
    if (!dims_ok(dims)) return 0;
    const MeasureGrid mg = measure_grid(dims);
    // + the list of active slices + the counter of the last reduction stage
    return ((size_t)dims[0] * 2 * mg.bpp * 2 + (size_t)dims[0] * 2) * sizeof(double) + kMaxNt * sizeof(uint16_t) + 16;
}

extern "C" int gf_init_lattice(gf_ctx** out, const int dims[4], int gauge, int recon, void* dev_links_f64,
                               void* dev_links_f32, void* dev_workspace, void* cuda_stream, uint64_t seed)
{
    if (!out) return GF_EINVAL;
    *out = nullptr;
    if (!dims_ok(dims)) return GF_EINVAL;
    if (gauge != GF_LANDAU && gauge != GF_COULOMB) return GF_EINVAL;
    if (recon != GF_RECON18 && recon != GF_RECON12) return GF_EINVAL;
    if (!dev_links_f64 && !dev_links_f32) return GF_EINVAL;
    if (!dev_workspace) return GF_EINVAL;
    if (((uintptr_t)dev_links_f64 | (uintptr_t)dev_links_f32 | (uintptr_t)dev_workspace) & 15u) return GF_EINVAL;

    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return GF_ECUDA;
    if (prop.major != 10) return GF_ECUDA;              // built for sm_100a only; no fallback

    gf_ctx* c = new (std::nothrow) gf_ctx;
    if (!c) return GF_ENOMEM;
    memset(c, 0, sizeof(*c));
    memcpy(c->dims, dims, sizeof(c->dims));
    c->gauge = gauge;
    c->recon = recon;
    c->links[PREC_F32] = dev_links_f32;
    c->links[PREC_F64] = dev_links_f64;
    c->device = dev;
    c->workspace = static_cast<double*>(dev_workspace);
    c->stream = static_cast<cudaStream_t>(cuda_stream);
    c->seed = seed;
    c->counter = 0;
    c->V = (size_t)dims[0] * dims[1] * dims[2] * dims[3];
    c->mg = measure_grid(dims);
    c->partials = c->workspace;
    c->slice_tmp = c->workspace + (size_t)dims[0] * 2 * c->mg.bpp * 2;
    c->dev_list = reinterpret_cast<uint16_t*>(c->slice_tmp + (size_t)dims[0] * 2);
    c->reduce_counter = reinterpret_cast<uint32_t*>(c->dev_list + kMaxNt);
    c->stop_dev = c->reduce_counter + 1;                 // both zeroed below
    c->runahead = 4;

    Geom& G = c->G;
    G.nt = dims[0];
    G.nxh = dims[1] / 2;
    G.ny = dims[2];
    G.nz = dims[3];
    G.Vh = (uint32_t)(c->V / 2);
    G.Vp[PREC_F32] = (G.Vh + Tile<float>::W - 1u) / Tile<float>::W * Tile<float>::W;
    G.Vp[PREC_F64] = (G.Vh + Tile<double>::W - 1u) / Tile<double>::W * Tile<double>::W;
    G.extent[0] = dims[0]; G.extent[1] = dims[1]; G.extent[2] = dims[2]; G.extent[3] = dims[3];
    G.stride[1] = 1;
    G.stride[2] = G.nxh;
    G.stride[3] = G.nxh * G.ny;
    G.stride[0] = G.nxh * G.ny * G.nz;
    G.div_nxh = make_fastdiv(G.nxh);
    G.div_ny = make_fastdiv(G.ny);
    G.div_nz = make_fastdiv(G.nz);
    G.sh = G.Vh / G.nt;
    G.div_sh = make_fastdiv(G.sh);

    // 0 = automatic (default_tuning below); gf_set_tuning overrides
    c->lanes[PREC_F32] = c->lanes[PREC_F64] = 0;
    c->block[PREC_F32] = c->block[PREC_F64] = 0;
    c->solver_mode = GF_SOLVER_AUTO;
    c->zigzag = 1;
    c->handoff = 1e-6;
    c->slab_rank = 0;
    c->slab_n = 1;

    if (cudaMemsetAsync(c->reduce_counter, 0, 16, c->stream) != cudaSuccess) {
        cudaGetLastError();
        delete c;
        return GF_ECUDA;
    }
    if (cudaMallocHost(reinterpret_cast<void**>(&c->host_pinned), sizeof(double) * 2 * kMaxNt + kMaxNt * (1 + sizeof(uint16_t)) + 16) != cudaSuccess) {
        cudaGetLastError();
        delete c;
        return GF_ENOMEM;
    }
    c->host_list = reinterpret_cast<uint16_t*>(c->host_pinned + 2 * kMaxNt);
    c->host_mask = reinterpret_cast<uint8_t*>(c->host_list + kMaxNt);
    for (int k = 0; k < kAsyncSlots; ++k) c->slot_precision[k] = -1;
    if (cudaMallocHost(reinterpret_cast<void**>(&c->host_slots), sizeof(double) * 2 * dims[0] * (kAsyncSlots + kRunAhead)) != cudaSuccess ||
        cudaHostGetDevicePointer(reinterpret_cast<void**>(&c->slots_dev), c->host_slots, 0) != cudaSuccess) {
        cudaGetLastError();
        if (c->host_slots) cudaFreeHost(c->host_slots);
        cudaFreeHost(c->host_pinned);
        delete c;
        return GF_ENOMEM;
    }
    if (cudaHostGetDevicePointer(reinterpret_cast<void**>(&c->slice_out), c->host_pinned, 0) != cudaSuccess) {
        cudaGetLastError();
        cudaFreeHost(c->host_slots);
        cudaFreeHost(c->host_pinned);
        delete c;
        return GF_ECUDA;
    }
    for (int k = 0; k < kRunAhead; ++k)
        if (cudaEventCreateWithFlags(&c->fix_events[k], cudaEventDisableTiming) != cudaSuccess) {
            cudaGetLastError();
            for (int j = 0; j < k; ++j) cudaEventDestroy(c->fix_events[j]);
            cudaFreeHost(c->host_slots);
            cudaFreeHost(c->host_pinned);
            delete c;
            return GF_ECUDA;
        }
    *out = c;
    return GF_OK;
}

extern "C" void gf_destroy(gf_ctx* ctx)
{
    if (!ctx) return;
    DeviceGuard guard(ctx);
    for (int k = 0; k < kRunAhead; ++k) cudaEventDestroy(ctx->fix_events[k]);
    if (ctx->host_pinned) cudaFreeHost(ctx->host_pinned);
    if (ctx->host_slots) cudaFreeHost(ctx->host_slots);
    delete ctx;
}

extern "C" const char* gf_last_error(const gf_ctx* ctx) { return ctx ? ctx->err : "null context"; }

static int check_prec(gf_ctx* ctx, int precision)
{
    if (!ctx) return GF_EINVAL;
    if (precision != GF_F32 && precision != GF_F64) return fail(ctx, GF_EINVAL, "precision must be GF_F32 or GF_F64");
    if (!ctx->links[precision]) return fail(ctx, GF_ESTATE, "no link storage for precision %d", precision);
    return GF_OK;
}

// Slab decomposition: every operation that reads or writes links is numbered; operation n of a slab
// starts when both neighbouring slabs have completed their operation n-1 (they may still be reading
// or writing the temporal links across the boundary), and publishes its completion.  The waits and
// writes are stream memory operations (no kernel spins, no host synchronisation).
static int slab_begin(gf_ctx* ctx)
{
    if (ctx->slab_n <= 1) return GF_OK;
    CUresult r = ctx->wait32((CUstream)ctx->stream, (CUdeviceptr)ctx->flag_prev, ctx->epoch, CU_STREAM_WAIT_VALUE_GEQ);
    if (r == CUDA_SUCCESS && ctx->flag_next != ctx->flag_prev)
        r = ctx->wait32((CUstream)ctx->stream, (CUdeviceptr)ctx->flag_next, ctx->epoch, CU_STREAM_WAIT_VALUE_GEQ);
    if (r != CUDA_SUCCESS) return fail(ctx, GF_ECUDA, "cuStreamWaitValue32 failed (%d)", (int)r);
    return GF_OK;
}

static int slab_end(gf_ctx* ctx)
{
    if (ctx->slab_n <= 1) return GF_OK;
    ctx->epoch += 1;
    CUresult r = ctx->write32((CUstream)ctx->stream, (CUdeviceptr)ctx->flag_own, ctx->epoch, CU_STREAM_WRITE_VALUE_DEFAULT);
    if (r != CUDA_SUCCESS) return fail(ctx, GF_ECUDA, "cuStreamWriteValue32 failed (%d)", (int)r);
    return GF_OK;
}

#define GF_SLAB_BEGIN(ctx)              \
    do {                                \
        int rc_ = slab_begin(ctx);      \
        if (rc_) return rc_;            \
    } while (0)
#define GF_SLAB_END(ctx)                \
    do {                                \
        int rc_ = slab_end(ctx);        \
        if (rc_) return rc_;            \
    } while (0)

// Slabs on different GPUs driven by one process: the kernels of this context dereference pointers into the
// neighbour's field, which needs peer access from this context's device to the neighbour's.
extern "C" int gf_enable_peer(gf_ctx* ctx, int peer_device)
{
    DeviceGuard guard(ctx);
    if (!ctx) return GF_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess) return cuda_fail(ctx, cudaGetLastError(), "gf_enable_peer");
    if (peer_device < 0 || peer_device >= ndev) return fail(ctx, GF_EINVAL, "no CUDA device %d", peer_device);
    if (peer_device == ctx->device) return GF_OK;
    int can = 0;
    cudaError_t e = cudaDeviceCanAccessPeer(&can, ctx->device, peer_device);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "gf_enable_peer");
    if (!can) return fail(ctx, GF_ECUDA, "device %d cannot access device %d as a peer", ctx->device, peer_device);
    e = cudaDeviceEnablePeerAccess(peer_device, 0);
    if (e == cudaErrorPeerAccessAlreadyEnabled) {
        cudaGetLastError();
        e = cudaSuccess;
    }
    if (e != cudaSuccess) return cuda_fail(ctx, e, "cudaDeviceEnablePeerAccess");
    return GF_OK;
}

extern "C" int gf_get_device(const gf_ctx* ctx, int* device_out)
{
    if (!ctx || !device_out) return GF_EINVAL;
    *device_out = ctx->device;
    return GF_OK;
}

extern "C" int gf_set_slab(gf_ctx* ctx, int rank, int nranks, void* dev_prev_links_f64, void* dev_prev_links_f32,
                           void* dev_next_links_f64, void* dev_next_links_f32, uint32_t* dev_flag_own,
                           uint32_t* dev_flag_prev, uint32_t* dev_flag_next)
{
    DeviceGuard guard(ctx);
    if (!ctx) return GF_EINVAL;
    if (nranks < 1 || rank < 0 || rank >= nranks) return fail(ctx, GF_EINVAL, "bad slab rank %d of %d", rank, nranks);
    if ((uint64_t)ctx->V * (uint64_t)nranks >= (uint64_t(1) << 32)) return fail(ctx, GF_EINVAL, "global volume must stay below 2^32 sites");
    if (nranks > 1) {
        if (!dev_flag_own || !dev_flag_prev || !dev_flag_next) return fail(ctx, GF_EINVAL, "slab flags missing");
        for (int prec = 0; prec < 2; ++prec) {
            void* pv = prec == PREC_F64 ? dev_prev_links_f64 : dev_prev_links_f32;
            void* nx = prec == PREC_F64 ? dev_next_links_f64 : dev_next_links_f32;
            if (ctx->links[prec] && (!pv || !nx)) return fail(ctx, GF_EINVAL, "neighbour fields missing for precision %d", prec);
            if (((uintptr_t)pv | (uintptr_t)nx) & 15u) return fail(ctx, GF_EINVAL, "neighbour fields must be 16-byte aligned");
        }
        if (ctx->gtrans[0] || ctx->gtrans[1] || ctx->defer_temporal)
            return fail(ctx, GF_ESTATE, "the transformation field and deferred temporal links are not available on slabs");
        if (!ctx->wait32) {
            cudaDriverEntryPointQueryResult q;
            void *w = nullptr, *wr = nullptr;
            if (cudaGetDriverEntryPoint("cuStreamWaitValue32", &w, cudaEnableDefault, &q) != cudaSuccess || !w ||
                cudaGetDriverEntryPoint("cuStreamWriteValue32", &wr, cudaEnableDefault, &q) != cudaSuccess || !wr) {
                cudaGetLastError();
                return fail(ctx, GF_ECUDA, "stream memory operations are not available");
            }
            ctx->wait32 = reinterpret_cast<decltype(ctx->wait32)>(w);
            ctx->write32 = reinterpret_cast<decltype(ctx->write32)>(wr);
        }
    }
    ctx->slab_rank = rank;
    ctx->slab_n = nranks;
    ctx->prev_links[PREC_F64] = nranks > 1 ? dev_prev_links_f64 : nullptr;
    ctx->prev_links[PREC_F32] = nranks > 1 ? dev_prev_links_f32 : nullptr;
    ctx->next_links[PREC_F64] = nranks > 1 ? dev_next_links_f64 : nullptr;
    ctx->next_links[PREC_F32] = nranks > 1 ? dev_next_links_f32 : nullptr;
    ctx->flag_own = dev_flag_own;
    ctx->flag_prev = dev_flag_prev;
    ctx->flag_next = dev_flag_next;
    ctx->epoch = 0;
    return GF_OK;
}

extern "C" int gf_pack(gf_ctx* ctx, const void* dev_canonical, int canonical_is_f64, int precision)
{
    DeviceGuard guard(ctx);
    int rc = check_prec(ctx, precision);
    if (rc) return rc;
    if (!dev_canonical) return fail(ctx, GF_EINVAL, "null canonical pointer");
    if ((uintptr_t)dev_canonical & 15u) return fail(ctx, GF_EINVAL, "the canonical buffer must be 16-byte aligned (it is read and written as 16-byte vectors)");
    ctx->pending[precision] = 0;      // the field is overwritten: nothing left to apply
    GF_SLAB_BEGIN(ctx);
    cudaError_t e = launch_pack(precision, ctx->recon, ctx->links[precision], ctx->G, dev_canonical, canonical_is_f64, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "gf_pack");
    GF_SLAB_END(ctx);
    ctx->launches += 1;
    return GF_OK;
}

extern "C" int gf_unpack(gf_ctx* ctx, void* dev_canonical, int canonical_is_f64, int precision)
{
    DeviceGuard guard(ctx);
    int rc = check_prec(ctx, precision);
    if (rc) return rc;
    rc = gf_coulomb_finish(ctx, precision);
    if (rc) return rc;
    if (!dev_canonical) return fail(ctx, GF_EINVAL, "null canonical pointer");
    if ((uintptr_t)dev_canonical & 15u) return fail(ctx, GF_EINVAL, "the canonical buffer must be 16-byte aligned (it is read and written as 16-byte vectors)");
    GF_SLAB_BEGIN(ctx);
    cudaError_t e = launch_unpack(precision, ctx->recon, ctx->links[precision], ctx->G, dev_canonical, canonical_is_f64, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "gf_unpack");
    GF_SLAB_END(ctx);
    ctx->launches += 1;
    return GF_OK;
}

static size_t canonical_bytes(const gf_ctx* ctx, int is_f64) { return ctx->V * 4 * 18 * (is_f64 ? 8 : 4); }

extern "C" int gf_load_host(gf_ctx* ctx, const void* host_canonical, int canonical_is_f64, int precision, void* dev_staging)
{
    DeviceGuard guard(ctx);
    int rc = check_prec(ctx, precision);
    if (rc) return rc;
    if (!host_canonical || !dev_staging) return fail(ctx, GF_EINVAL, "null host or staging pointer");
    if ((uintptr_t)dev_staging & 15u) return fail(ctx, GF_EINVAL, "the staging buffer must be 16-byte aligned (it is read and written as 16-byte vectors)");
    cudaError_t e = cudaMemcpyAsync(dev_staging, host_canonical, canonical_bytes(ctx, canonical_is_f64), cudaMemcpyHostToDevice, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "gf_load_host copy");
    return gf_pack(ctx, dev_staging, canonical_is_f64, precision);
}

extern "C" int gf_store_host(gf_ctx* ctx, void* host_canonical, int canonical_is_f64, int precision, void* dev_staging)
{
    DeviceGuard guard(ctx);
    int rc = check_prec(ctx, precision);
    if (rc) return rc;
    if (!host_canonical || !dev_staging) return fail(ctx, GF_EINVAL, "null host or staging pointer");
    if ((uintptr_t)dev_staging & 15u) return fail(ctx, GF_EINVAL, "the staging buffer must be 16-byte aligned (it is read and written as 16-byte vectors)");
    rc = gf_unpack(ctx, dev_staging, canonical_is_f64, precision);
    if (rc) return rc;
    cudaError_t e = cudaMemcpyAsync(host_canonical, dev_staging, canonical_bytes(ctx, canonical_is_f64), cudaMemcpyDeviceToHost, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "gf_store_host copy");
    return sync_and_check(ctx, "gf_store_host copy");
}

static int check_algo(gf_ctx* ctx, int algo, double omega, double p)
{
    if (algo != GF_RELAX && algo != GF_OVERRELAX && algo != GF_STOCHASTIC) return fail(ctx, GF_EINVAL, "unknown algo %d", algo);
    if (algo == GF_OVERRELAX && !(omega >= 1.0 && omega < 2.0)) return fail(ctx, GF_EINVAL, "omega must be in [1,2)");
    if (algo == GF_STOCHASTIC && !(p >= 0.0 && p <= 1.0)) return fail(ctx, GF_EINVAL, "p must be in [0,1]");
    return GF_OK;
}

// Launch configuration chosen by measurement on B200 at 32^4 (profiles/r2_tune_f64_12.txt, profiles/r3_tune_solver.txt,
// DESIGN.md "Kernels"): two lanes per site everywhere except fp64 / 12-real, where one lane per site (no redundant
// solve, third rows never held in registers) is the variant that stays bandwidth-bound under the power cap.
static void default_tuning(int precision, int recon, int solver_f64, int accumulate, int defer, uint32_t Vh, int* lanes, int* block)
{
    // Lattices of less than one wave of blocks are bound by the latency of a single site update, not by bandwidth: more
    // lanes per site shorten it (8^4: 9.2 instead of 12.3 us per fp64 / 12-real iteration; 16^4 fp32 / 12-real: 12.3
    // instead of 16.4 us with two lanes).
    if (Vh <= 4096u) {
        *lanes = 4;
        *block = 64;
        return;
    }
    if (Vh <= 65536u && precision == GF_F32 && recon == GF_RECON12 && !solver_f64 && !defer) {
        *lanes = 2;
        *block = 64;
        return;
    }
    if (defer && precision == GF_F32) {      // 6 links + G: one lane per site is balanced and fits the registers
        *lanes = 1;
        *block = 64;
        return;
    }
    if (precision == GF_F64) {
        *lanes = recon == GF_RECON12 ? 1 : 2;
        *block = recon == GF_RECON12 ? 64 : 128;
    } else {
        *lanes = 2;
        *block = (recon == GF_RECON18 && !solver_f64) ? 128 : 64;
        if (recon == GF_RECON12 && !solver_f64) *lanes = 1;     // tiled layout: 100 % against 96 % with two lanes (profiles/r2_tune_f32_12.txt)
        // fp64-register solver (the default): 18-real is best with one lane per site (97.5 % against 94.7 % at 32^4, 69.5 %
        // against 63.2 % at 16^4), 12-real with two (83.8 % against 80.2 %): profiles/r3_tune_solver.txt
        if (recon == GF_RECON18 && solver_f64 && !accumulate) *lanes = 1;
    }
}

static int enqueue_sweep(gf_ctx* ctx, int parity, int algo, double omega, double p, int precision)
{
    if (ctx->defer_temporal) {
        if (!ctx->gtrans[precision])
            return fail(ctx, GF_ESTATE, "deferred temporal links need a transformation buffer for precision %d (gf_set_transform)", precision);
        if (!ctx->pending[precision]) {      // G(x) restarts from the identity: it is what gf_coulomb_finish will apply
            int rc = write_identity(ctx, precision);
            if (rc) return rc;
            ctx->pending[precision] = 1;
        }
    }
    SweepArgs a;
    memset(&a, 0, sizeof(a));
    a.links = ctx->links[precision];
    a.gtrans = ctx->gtrans[precision];
    a.defer_temporal = ctx->defer_temporal;
    a.slice_list = ctx->mask_on ? ctx->dev_list : nullptr;
    a.n_listed = (uint32_t)ctx->n_active;
    a.prev_links = ctx->prev_links[precision];
    a.site_offset = (uint32_t)((uint64_t)ctx->slab_rank * ctx->V);
    a.G = ctx->G;
    a.parity = (uint32_t)parity;
    a.mu0 = ctx->gauge == GF_COULOMB ? 1 : 0;
    a.algo = algo;
    a.omega = omega;
    a.p = p;
    a.key0 = (uint32_t)ctx->seed;
    a.key1 = (uint32_t)(ctx->seed >> 32);
    a.counter = ctx->counter;
    a.reverse = ctx->zigzag ? (uint32_t)(ctx->sweeps & 1u) : 0u;
    a.stop = ctx->stop_dev;
    // fp32 storage: K(x) and the SU(2) solves in fp64 registers unless the caller asked for fp32 (gf_set_solver_precision).
    // The all-fp32 solve amplifies its rounding by |K| / |v| at sites whose SU(2) projection is small: one site in 5 x 10^5
    // of the 32^4 bench field ends 1.08e-5 from the oracle after one iteration, above north_star's 1e-5.
    const int solver_f64 = ctx->solver_mode == GF_SOLVER_AUTO ? 1 : ctx->solver_mode == GF_F64;
    (void)algo;
    int lanes, block;
    default_tuning(precision, ctx->recon, solver_f64, a.gtrans != nullptr, a.gtrans != nullptr && a.defer_temporal, ctx->G.Vh, &lanes, &block);
    if (ctx->lanes[precision]) lanes = ctx->lanes[precision];
    if (ctx->block[precision]) block = ctx->block[precision];
    if (a.slice_list && a.n_listed == 0) {   // every slice frozen: the half-sweep is empty, the Philox counter still advances
        ctx->counter += 1;
        return GF_OK;
    }
    GF_SLAB_BEGIN(ctx);
    cudaError_t e = launch_sweep(precision, solver_f64, ctx->recon, lanes, block, a, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "gf_sweep launch");
    GF_SLAB_END(ctx);
    ctx->counter += 1;
    ctx->sweeps += 1;
    ctx->launches += 1;
    return GF_OK;
}

// One iteration = parity 0 then parity 1.
static int enqueue_iteration(gf_ctx* ctx, int algo, double omega, double p, int precision)
{
    int e = enqueue_sweep(ctx, 0, algo, omega, p, precision);
    if (e == GF_OK) e = enqueue_sweep(ctx, 1, algo, omega, p, precision);
    return e;
}

extern "C" int gf_iterate(gf_ctx* ctx, int n, int algo, double omega, double p, int precision)
{
    DeviceGuard guard(ctx);
    int rc = check_prec(ctx, precision);
    if (rc) return rc;
    if (n < 0) return fail(ctx, GF_EINVAL, "negative iteration count");
    rc = check_algo(ctx, algo, omega, p);
    if (rc) return rc;
    for (int k = 0; k < n; ++k) {
        rc = enqueue_iteration(ctx, algo, omega, p, precision);
        if (rc) return rc;
    }
    return GF_OK;
}

extern "C" int gf_sweep(gf_ctx* ctx, int parity, int algo, double omega, double p, int precision)
{
    DeviceGuard guard(ctx);
    int rc = check_prec(ctx, precision);
    if (rc) return rc;
    if (parity != 0 && parity != 1) return fail(ctx, GF_EINVAL, "parity must be 0 or 1");
    rc = check_algo(ctx, algo, omega, p);
    if (rc) return rc;
    return enqueue_sweep(ctx, parity, algo, omega, p, precision);
}

// Last reduction stage of F / theta: Landau 1/(Nc Nd V) and 1/(Nc V) over the whole lattice (on slabs:
// this slab's share of the global sums, the caller adds the slabs up); Coulomb per slice 1/(Nc 3 Ns^3) and 1/(Nc Ns^3).
static ReduceTail measure_tail(const gf_ctx* ctx)
{
    ReduceTail t;
    t.slice_tmp = ctx->slice_tmp;
    t.counter = ctx->reduce_counter;
    t.stop = nullptr;
    t.target = 0.0;
    t.stall = 0.0;
    t.prev = nullptr;
    if (ctx->gauge == GF_COULOMB) {
        const double Vs = (double)(ctx->V / ctx->dims[0]);
        t.combine = 0;
        t.scale0 = 1.0 / (3.0 * 3.0 * Vs);
        t.scale1 = 1.0 / (3.0 * Vs);
    } else {
        t.combine = 1;
        t.scale0 = 1.0 / (3.0 * 4.0 * (double)ctx->V * ctx->slab_n);
        t.scale1 = 1.0 / (3.0 * (double)ctx->V * ctx->slab_n);
    }
    return t;
}

static ReduceTail lattice_tail(const gf_ctx* ctx, double scale)
{
    ReduceTail t;
    t.slice_tmp = ctx->slice_tmp;
    t.counter = ctx->reduce_counter;
    t.combine = 1;
    t.scale0 = t.scale1 = scale;
    t.stop = nullptr;
    t.target = 0.0;
    t.stall = 0.0;
    t.prev = nullptr;
    return t;
}

static int sync_and_check(gf_ctx* ctx, const char* what)
{
    cudaError_t e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, what);
    return GF_OK;
}

// Runs the measurement kernels and leaves F and theta (Coulomb: per slice, interleaved) in ctx->host_pinned.
// active_only (the fix loop with slice freezing): only the slices still being swept are measured; the frozen ones keep
// the F_t, theta_t of their last evaluation in host_pinned -- nothing that enters them has changed since.
static int measure_to_host(gf_ctx* ctx, int precision, bool active_only = false)
{
    const int mu0 = ctx->gauge == GF_COULOMB ? 1 : 0;
    MeasureGrid mg = ctx->mg;
    if (active_only && ctx->mask_on && ctx->gauge == GF_COULOMB) {
        if (ctx->n_active == 0) return GF_OK;
        mg.slice_list = ctx->dev_list;
        mg.n_listed = (uint32_t)ctx->n_active;
    }
    GF_SLAB_BEGIN(ctx);
    cudaError_t e = launch_measure(precision, ctx->recon, ctx->links[precision], ctx->prev_links[precision], ctx->G, mu0, mg,
                                   ctx->partials, measure_tail(ctx), ctx->slice_out, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "measure launch");
    GF_SLAB_END(ctx);
    ctx->launches += 2;
    return sync_and_check(ctx, "measure");
}

// Copies the results the reduction kernels left in (mapped) host memory: Landau (F, theta), Coulomb (F_t, theta_t)
// per slice.  Returns theta, in Coulomb gauge max_t theta_t -- what the fix loop compares with its target.
static double finish_measure(const gf_ctx* ctx, double* host_F, double* host_theta, const double* sums = nullptr)
{
    const double* s = sums ? sums : ctx->host_pinned;
    if (ctx->gauge != GF_COULOMB) {
        if (host_F) host_F[0] = s[0];
        if (host_theta) host_theta[0] = s[1];
        return s[1];
    }
    double worst = 0.0;
    for (int t = 0; t < ctx->dims[0]; ++t) {
        if (host_F) host_F[t] = s[2 * t];
        if (host_theta) host_theta[t] = s[2 * t + 1];
        if (s[2 * t + 1] > worst || t == 0) worst = s[2 * t + 1];
    }
    return worst;
}

extern "C" int gf_measure(gf_ctx* ctx, int precision, double* host_functional, double* host_theta)
{
    DeviceGuard guard(ctx);
    int rc = check_prec(ctx, precision);
    if (rc) return rc;
    rc = measure_to_host(ctx, precision);
    if (rc) return rc;
    finish_measure(ctx, host_functional, host_theta);
    return GF_OK;
}

extern "C" int gf_measure_async(gf_ctx* ctx, int precision, int slot)
{
    DeviceGuard guard(ctx);
    int rc = check_prec(ctx, precision);
    if (rc) return rc;
    if (slot < 0 || slot >= kAsyncSlots) return fail(ctx, GF_EINVAL, "slot must be 0..%d", kAsyncSlots - 1);
    const int mu0 = ctx->gauge == GF_COULOMB ? 1 : 0;
    GF_SLAB_BEGIN(ctx);
    cudaError_t e = launch_measure(precision, ctx->recon, ctx->links[precision], ctx->prev_links[precision], ctx->G, mu0, ctx->mg,
                                   ctx->partials, measure_tail(ctx), ctx->slots_dev + (size_t)slot * 2 * ctx->dims[0], ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "measure launch");
    GF_SLAB_END(ctx);
    ctx->launches += 2;
    ctx->slot_precision[slot] = precision;
    return GF_OK;
}

extern "C" int gf_measure_collect(gf_ctx* ctx, int slot, double* host_functional, double* host_theta)
{
    DeviceGuard guard(ctx);
    if (!ctx) return GF_EINVAL;
    if (slot < 0 || slot >= kAsyncSlots) return fail(ctx, GF_EINVAL, "slot must be 0..%d", kAsyncSlots - 1);
    if (ctx->slot_precision[slot] < 0) return fail(ctx, GF_ESTATE, "nothing was measured into slot %d", slot);
    int rc = sync_and_check(ctx, "gf_measure_collect");
    if (rc) return rc;
    finish_measure(ctx, host_functional, host_theta, ctx->host_slots + (size_t)slot * 2 * ctx->dims[0]);
    ctx->slot_precision[slot] = -1;
    return GF_OK;
}

extern "C" int gf_functional(gf_ctx* ctx, int precision, double* host_out)
{
    DeviceGuard guard(ctx);
    if (ctx && !host_out) return fail(ctx, GF_EINVAL, "null output");
    return gf_measure(ctx, precision, host_out, nullptr);
}

extern "C" int gf_theta(gf_ctx* ctx, int precision, double* host_out)
{
    DeviceGuard guard(ctx);
    if (ctx && !host_out) return fail(ctx, GF_EINVAL, "null output");
    return gf_measure(ctx, precision, nullptr, host_out);
}

// Re-projection of the field being swept (and of the transformation recorded with it) onto SU(3) inside a fix loop
// (gf_set_reunitarize_every): Gram-Schmidt on rows 0 and 1 in fp64, row 2 rebuilt.  Enqueued at an evaluation point, before
// theta is measured; `stop`: the run-ahead loop's stop word (the re-projection too must leave a converged field alone).
static int enqueue_reunitarize(gf_ctx* ctx, int precision, const uint32_t* stop)
{
    cudaError_t e = launch_cast(precision, precision, ctx->recon, ctx->links[precision], ctx->links[precision], ctx->G, 1, 8, ctx->stream, stop);
    if (e == cudaSuccess && ctx->gtrans[precision]) {
        e = launch_cast(precision, precision, ctx->recon, ctx->gtrans[precision], ctx->gtrans[precision], ctx->G, 1, 2, ctx->stream, stop);
        ctx->launches += 1;
    }
    if (e != cudaSuccess) return cuda_fail(ctx, e, "re-projection in the fix loop");
    ctx->launches += 1;
    return GF_OK;
}

// The fix loop without a host round trip per evaluation.  Blocks of {iterations up to the next evaluation; F / theta
// reduction} are enqueued up to ctx->runahead ahead of the block whose result the host is waiting for.  The last
// reduction kernel of a block compares theta with the target ON THE DEVICE (the same double, the same comparison the
// host makes when it reads the value from pinned memory) and sets ctx->stop_dev; the half-sweeps already enqueued
// behind it then leave the field alone.  The host reads the blocks in order, stops at the first one below the target
// and rewinds its half-sweep counter to that block: field, iteration count and Philox stream are those of the loop
// that waits for every theta (fix_phase below with runahead = 0).
static int fix_phase_runahead(gf_ctx* ctx, int algo, double omega, double p, int precision, double target, int max_iter,
                              int check_every, int* it_io, double* theta_out, double stall)
{
    struct Block { int it_end; uint32_t counter_end; uint64_t sweeps_end; } meta[kRunAhead];
    const int depth = ctx->runahead < kRunAhead ? ctx->runahead : kRunAhead;
    const int mu0 = ctx->gauge == GF_COULOMB ? 1 : 0;
    const size_t slot_len = (size_t)2 * ctx->dims[0];
    int it_enq = *it_io, rc = GF_NOT_CONVERGED, err = GF_OK, since_reunit = 0;
    long head = 0, tail = 0;
    ReduceTail rt = measure_tail(ctx);
    rt.stop = ctx->stop_dev;
    rt.target = target;
    rt.stall = stall;
    rt.prev = reinterpret_cast<double*>(ctx->reduce_counter + 2);      // third and fourth word of the 16 bytes: 8-byte aligned
    double prev_theta = 0.0;
    if (stall > 0.0) {
        cudaError_t e0 = cudaMemsetAsync(rt.prev, 0, sizeof(double), ctx->stream);
        if (e0 != cudaSuccess) return cuda_fail(ctx, e0, "fix loop");
    }
    while (true) {
        while (err == GF_OK && head - tail < depth && it_enq < max_iter) {
            int n = check_every - (it_enq % check_every);
            if (n > max_iter - it_enq) n = max_iter - it_enq;
            for (int k = 0; k < n && err == GF_OK; ++k) err = enqueue_iteration(ctx, algo, omega, p, precision);
            if (err != GF_OK) break;
            it_enq += n;
            since_reunit += n;
            if (ctx->reunit_every > 0 && since_reunit >= ctx->reunit_every) {
                err = enqueue_reunitarize(ctx, precision, ctx->stop_dev);
                if (err != GF_OK) break;
                since_reunit = 0;
            }
            const int s = (int)(head % depth);
            cudaError_t e = launch_measure(precision, ctx->recon, ctx->links[precision], ctx->prev_links[precision], ctx->G, mu0,
                                           ctx->mg, ctx->partials, rt, ctx->slots_dev + (size_t)(kAsyncSlots + s) * slot_len, ctx->stream);
            if (e == cudaSuccess) e = cudaEventRecord(ctx->fix_events[s], ctx->stream);
            if (e != cudaSuccess) { err = cuda_fail(ctx, e, "fix loop"); break; }
            ctx->launches += 2;
            meta[s].it_end = it_enq;
            meta[s].counter_end = ctx->counter;
            meta[s].sweeps_end = ctx->sweeps;
            ++head;
        }
        if (tail == head) break;                        // nothing in flight: max_iter reached (or an error before any block)
        const int s = (int)(tail % depth);
        cudaError_t e = cudaEventSynchronize(ctx->fix_events[s]);
        if (e != cudaSuccess) { err = cuda_fail(ctx, e, "fix loop"); break; }
        *theta_out = finish_measure(ctx, nullptr, nullptr, ctx->host_slots + (size_t)(kAsyncSlots + s) * slot_len);
        *it_io = meta[s].it_end;
        ++tail;
        const bool stalled = stall > 0.0 && prev_theta > 0.0 && *theta_out >= stall * prev_theta;
        prev_theta = *theta_out;
        if (*theta_out < target || stalled) {
            // the device took the same decision after this block: what is enqueued behind it is a no-op there
            ctx->counter = meta[s].counter_end;
            ctx->sweeps = meta[s].sweeps_end;
            rc = *theta_out < target ? GF_OK : GF_NOT_CONVERGED;
            break;
        }
    }
    // behind everything enqueued so far: later sweeps of this context act again
    cudaError_t e = cudaMemsetAsync(ctx->stop_dev, 0, sizeof(uint32_t), ctx->stream);
    if (e != cudaSuccess && err == GF_OK) err = cuda_fail(ctx, e, "fix loop");
    return err != GF_OK ? err : rc;
}

// One phase of the fix loop in one precision.  Returns GF_OK when theta < target was seen.
// stall > 0 (fp32 phase of the mixed-precision runs): the phase also ends, with GF_NOT_CONVERGED, at the first evaluation
// whose theta is not below stall * (theta of the previous evaluation).
static int fix_phase(gf_ctx* ctx, int algo, double omega, double p, int precision, double target, int max_iter,
                     int check_every, int* it_io, double* theta_out, double stall = 0.0)
{
    int it = *it_io, since_reunit = 0;
    double prev_theta = 0.0;
    int rc = GF_NOT_CONVERGED;
    const bool freeze = ctx->freeze_slices && ctx->gauge == GF_COULOMB;
    // slice freezing changes the launch list between evaluations on the host: that loop waits for every theta
    if (!freeze && ctx->runahead > 0) return fix_phase_runahead(ctx, algo, omega, p, precision, target, max_iter, check_every, it_io, theta_out, stall);
    if (freeze) {                            // every slice starts active (the stream is idle or ordered: pinned copy is free)
        cudaError_t e = cudaStreamSynchronize(ctx->stream);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "fix loop");
        for (int t = 0; t < ctx->dims[0]; ++t) ctx->host_mask[t] = 1;
        ctx->mask_on = 1;
        int rc0 = upload_mask(ctx);
        if (rc0) return rc0;
    }
    while (it < max_iter) {
        int n = check_every - (it % check_every);
        if (n > max_iter - it) n = max_iter - it;
        for (int k = 0; k < n; ++k) {
            int e = enqueue_iteration(ctx, algo, omega, p, precision);
            if (e != GF_OK) { *it_io = it; if (freeze) ctx->mask_on = 0; return e; }
        }
        it += n;
        since_reunit += n;
        if (ctx->reunit_every > 0 && since_reunit >= ctx->reunit_every) {
            int er = enqueue_reunitarize(ctx, precision, nullptr);
            if (er != GF_OK) { *it_io = it; if (freeze) ctx->mask_on = 0; return er; }
            since_reunit = 0;
        }
        int e = measure_to_host(ctx, precision, freeze);
        if (e != GF_OK) { *it_io = it; if (freeze) ctx->mask_on = 0; return e; }
        *theta_out = finish_measure(ctx, nullptr, nullptr);
        if (*theta_out < target) { rc = GF_OK; break; }
        if (stall > 0.0 && prev_theta > 0.0 && *theta_out >= stall * prev_theta) break;
        prev_theta = *theta_out;
        if (freeze) {
            // reading A17b: a slice below the target stops being swept; nothing that enters its F_t and
            // theta_t changes afterwards, so max_t theta_t above remains the stopping criterion
            bool changed = false;
            for (int t = 0; t < ctx->dims[0]; ++t)
                if (ctx->host_mask[t] && ctx->host_pinned[2 * t + 1] < target) {
                    ctx->host_mask[t] = 0;
                    changed = true;
                }
            if (changed) {
                e = upload_mask(ctx);
                if (e != GF_OK) { *it_io = it; ctx->mask_on = 0; return e; }
            }
        }
    }
    if (freeze) ctx->mask_on = 0;
    *it_io = it;
    return rc;
}

// Second phase of the mixed-precision runs.  The fp64 field has just been produced from the fp32 phase (cast +
// re-projection, or the replayed transformation): theta is re-measured on IT -- the value returned always
// refers to the fp64 result, never to the fp32 field -- and the fp64 iterations run while it is above the
// target and iterations are left.
static int finish_in_f64(gf_ctx* ctx, int algo, double omega, double p, double target, int max_iter, int check_every,
                         int* it_io, double* theta_out)
{
    int e = measure_to_host(ctx, GF_F64);
    if (e != GF_OK) return e;
    *theta_out = finish_measure(ctx, nullptr, nullptr);
    if (*theta_out < target) return GF_OK;
    if (*it_io >= max_iter) return GF_NOT_CONVERGED;
    return fix_phase(ctx, algo, omega, p, GF_F64, target, max_iter, check_every, it_io, theta_out);
}

extern "C" int gf_fix_until(gf_ctx* ctx, int algo, double omega, double p, int precision, double theta_target,
                            int max_iter, int check_every, int* iters_out, double* theta_out)
{
    DeviceGuard guard(ctx);
    if (!ctx) return GF_EINVAL;
    const bool mixed = precision == GF_MIXED || precision == GF_MIXED_EXACT;
    if (precision != GF_F32 && precision != GF_F64 && !mixed) return fail(ctx, GF_EINVAL, "bad precision");
    if (mixed && (!ctx->links[PREC_F32] || !ctx->links[PREC_F64]))
        return fail(ctx, GF_ESTATE, "GF_MIXED / GF_MIXED_EXACT need both fp32 and fp64 storage");
    if (precision == GF_MIXED_EXACT && (!ctx->gtrans[PREC_F32] || !ctx->gtrans[PREC_F64]))
        return fail(ctx, GF_ESTATE, "GF_MIXED_EXACT needs both transformation buffers (gf_set_transform)");
    if (!mixed && !ctx->links[precision]) return fail(ctx, GF_ESTATE, "no link storage for precision %d", precision);
    int rc = check_algo(ctx, algo, omega, p);
    if (rc) return rc;
    if (max_iter < 0 || check_every < 1 || !(theta_target >= 0.0)) return fail(ctx, GF_EINVAL, "bad max_iter / check_every / theta_target");
    if (ctx->slab_n > 1) return fail(ctx, GF_ESTATE, "gf_fix_until needs the whole lattice: on slabs the caller runs the loop and adds up theta");
    if (ctx->defer_temporal && precision == GF_MIXED_EXACT)
        return fail(ctx, GF_ESTATE, "GF_MIXED_EXACT and deferred temporal links both use the transformation buffers");
    if (ctx->defer_temporal && ((precision != GF_F64 && !ctx->gtrans[PREC_F32]) || (precision != GF_F32 && !ctx->gtrans[PREC_F64])))
        return fail(ctx, GF_ESTATE, "deferred temporal links need a transformation buffer for every precision swept (gf_set_transform)");

    int it = 0;
    double theta = -1.0;
    if (precision == GF_MIXED) {
        const double t32 = theta_target > ctx->handoff ? theta_target : ctx->handoff;
        rc = fix_phase(ctx, algo, omega, p, GF_F32, t32, max_iter, check_every, &it, &theta, ctx->stall);
        if (rc < 0) return rc;
        int e = gf_cast(ctx, GF_F32, GF_F64);
        if (e != GF_OK) return e;
        rc = finish_in_f64(ctx, algo, omega, p, theta_target, max_iter, check_every, &it, &theta);
    } else if (precision == GF_MIXED_EXACT) {
        // fp32 sweeps on a copy, recording G(x); then the untouched fp64 input is transformed by the
        // re-projected G (gauge equivalent to the input at fp64 accuracy) and the fp64 phase goes on
        // accumulating into the fp64 transformation.
        int e = gf_cast(ctx, GF_F64, GF_F32);
        if (e == GF_OK) e = gf_transform_identity(ctx, GF_F32);
        if (e != GF_OK) return e;
        const double t32 = theta_target > ctx->handoff ? theta_target : ctx->handoff;
        rc = fix_phase(ctx, algo, omega, p, GF_F32, t32, max_iter, check_every, &it, &theta, ctx->stall);
        if (rc < 0) return rc;
        e = gf_transform_cast(ctx, GF_F32, GF_F64);
        if (e == GF_OK) e = gf_apply_transform(ctx, GF_F64, GF_F64, GF_F64);
        if (e != GF_OK) return e;
        rc = finish_in_f64(ctx, algo, omega, p, theta_target, max_iter, check_every, &it, &theta);
    } else {
        if (max_iter == 0) {
            rc = measure_to_host(ctx, precision);
            if (rc) return rc;
            theta = finish_measure(ctx, nullptr, nullptr);
            rc = theta < theta_target ? GF_OK : GF_NOT_CONVERGED;
        } else {
            rc = fix_phase(ctx, algo, omega, p, precision, theta_target, max_iter, check_every, &it, &theta);
        }
    }
    if (rc < 0) return rc;
    for (int prec = 0; prec < 2; ++prec) {          // deferred temporal links: the result is a complete field
        int e = gf_coulomb_finish(ctx, prec);
        if (e != GF_OK) return e;
    }
    if (iters_out) *iters_out = it;
    if (theta_out) *theta_out = theta;
    return rc;
}

extern "C" int gf_set_rng(gf_ctx* ctx, uint64_t seed, uint32_t half_sweep_counter)
{
    DeviceGuard guard(ctx);
    if (!ctx) return GF_EINVAL;
    ctx->seed = seed;
    ctx->counter = half_sweep_counter;
    return GF_OK;
}

extern "C" int gf_get_counter(const gf_ctx* ctx, uint32_t* half_sweep_counter_out)
{
    if (!ctx || !half_sweep_counter_out) return GF_EINVAL;
    *half_sweep_counter_out = ctx->counter;
    return GF_OK;
}

extern "C" int gf_reunitarize(gf_ctx* ctx, int precision)
{
    DeviceGuard guard(ctx);
    int rc = check_prec(ctx, precision);
    if (rc) return rc;
    rc = gf_coulomb_finish(ctx, precision);
    if (rc) return rc;
    GF_SLAB_BEGIN(ctx);
    cudaError_t e = launch_cast(precision, precision, ctx->recon, ctx->links[precision], ctx->links[precision], ctx->G, 1, 8, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "gf_reunitarize");
    GF_SLAB_END(ctx);
    ctx->launches += 1;
    return GF_OK;
}

extern "C" int gf_cast(gf_ctx* ctx, int from_precision, int to_precision)
{
    DeviceGuard guard(ctx);
    int rc = check_prec(ctx, from_precision);
    if (rc) return rc;
    rc = check_prec(ctx, to_precision);
    if (rc) return rc;
    if (from_precision == to_precision) return fail(ctx, GF_EINVAL, "gf_cast needs two different precisions");
    rc = gf_coulomb_finish(ctx, from_precision);
    if (rc) return rc;
    ctx->pending[to_precision] = 0;   // the destination field is overwritten: nothing left to apply to it
    const int reproject = from_precision == GF_F32 && to_precision == GF_F64;
    GF_SLAB_BEGIN(ctx);
    cudaError_t e = launch_cast(from_precision, to_precision, ctx->recon, ctx->links[from_precision], ctx->links[to_precision],
                                ctx->G, reproject, 8, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "gf_cast");
    GF_SLAB_END(ctx);
    ctx->launches += 1;
    return GF_OK;
}

// ---------------------------------------------------------- the accumulated transformation
extern "C" int gf_set_transform(gf_ctx* ctx, void* dev_g_f64, void* dev_g_f32)
{
    DeviceGuard guard(ctx);
    if (!ctx) return GF_EINVAL;
    if (((uintptr_t)dev_g_f64 | (uintptr_t)dev_g_f32) & 15u) return fail(ctx, GF_EINVAL, "transformation buffers must be 16-byte aligned");
    if (ctx->slab_n > 1 && (dev_g_f64 || dev_g_f32)) return fail(ctx, GF_ESTATE, "the transformation field is not available on slabs");
    if ((ctx->pending[PREC_F64] && dev_g_f64 != ctx->gtrans[PREC_F64]) || (ctx->pending[PREC_F32] && dev_g_f32 != ctx->gtrans[PREC_F32]))
        return fail(ctx, GF_ESTATE, "a transformation buffer holds a deferred temporal update: call gf_coulomb_finish before replacing it");
    ctx->gtrans[PREC_F64] = dev_g_f64;
    ctx->gtrans[PREC_F32] = dev_g_f32;
    return GF_OK;
}

static int check_transform(gf_ctx* ctx, int precision)
{
    if (!ctx) return GF_EINVAL;
    if (precision != GF_F32 && precision != GF_F64) return fail(ctx, GF_EINVAL, "precision must be GF_F32 or GF_F64");
    if (!ctx->gtrans[precision]) return fail(ctx, GF_ESTATE, "no transformation buffer for precision %d (gf_set_transform)", precision);
    return GF_OK;
}

// While a deferred temporal update is outstanding (gf_set_coulomb_mode) the transformation buffer holds the only
// copy of what still has to be applied to U_0: nothing may overwrite it before gf_coulomb_finish.
static int check_transform_writable(gf_ctx* ctx, int precision)
{
    int rc = check_transform(ctx, precision);
    if (rc) return rc;
    if (ctx->pending[precision])
        return fail(ctx, GF_ESTATE, "the transformation buffer of precision %d holds a deferred temporal update: call gf_coulomb_finish first",
                    precision);
    return GF_OK;
}

static int write_identity(gf_ctx* ctx, int precision)
{
    cudaError_t e = launch_transform_identity(precision, ctx->recon, ctx->gtrans[precision], ctx->G, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "gf_transform_identity");
    ctx->launches += 1;
    return GF_OK;
}

extern "C" int gf_transform_identity(gf_ctx* ctx, int precision)
{
    DeviceGuard guard(ctx);
    int rc = check_transform_writable(ctx, precision);
    if (rc) return rc;
    return write_identity(ctx, precision);
}

extern "C" int gf_transform_pack(gf_ctx* ctx, const void* dev_canonical, int canonical_is_f64, int precision)
{
    DeviceGuard guard(ctx);
    int rc = check_transform_writable(ctx, precision);
    if (rc) return rc;
    if (!dev_canonical) return fail(ctx, GF_EINVAL, "null canonical pointer");
    if ((uintptr_t)dev_canonical & 15u) return fail(ctx, GF_EINVAL, "the canonical buffer must be 16-byte aligned (it is read and written as 16-byte vectors)");
    cudaError_t e = launch_transform_pack(precision, ctx->recon, ctx->gtrans[precision], ctx->G, dev_canonical, canonical_is_f64, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "gf_transform_pack");
    ctx->launches += 1;
    return GF_OK;
}

extern "C" int gf_transform_unpack(gf_ctx* ctx, void* dev_canonical, int canonical_is_f64, int precision)
{
    DeviceGuard guard(ctx);
    int rc = check_transform(ctx, precision);
    if (rc) return rc;
    if (!dev_canonical) return fail(ctx, GF_EINVAL, "null canonical pointer");
    if ((uintptr_t)dev_canonical & 15u) return fail(ctx, GF_EINVAL, "the canonical buffer must be 16-byte aligned (it is read and written as 16-byte vectors)");
    cudaError_t e = launch_transform_unpack(precision, ctx->recon, ctx->gtrans[precision], ctx->G, dev_canonical, canonical_is_f64, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "gf_transform_unpack");
    ctx->launches += 1;
    return GF_OK;
}

extern "C" int gf_transform_cast(gf_ctx* ctx, int from_precision, int to_precision)
{
    DeviceGuard guard(ctx);
    int rc = check_transform(ctx, from_precision);
    if (rc) return rc;
    rc = check_transform_writable(ctx, to_precision);
    if (rc) return rc;
    if (from_precision == to_precision) return fail(ctx, GF_EINVAL, "gf_transform_cast needs two different precisions");
    const int reproject = from_precision == GF_F32 && to_precision == GF_F64;
    cudaError_t e = launch_cast(from_precision, to_precision, ctx->recon, ctx->gtrans[from_precision], ctx->gtrans[to_precision],
                                ctx->G, reproject, 2, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "gf_transform_cast");
    ctx->launches += 1;
    return GF_OK;
}

extern "C" int gf_apply_transform(gf_ctx* ctx, int g_precision, int src_precision, int dst_precision)
{
    DeviceGuard guard(ctx);
    int rc = check_transform(ctx, g_precision);
    if (rc) return rc;
    rc = check_prec(ctx, src_precision);
    if (rc) return rc;
    rc = check_prec(ctx, dst_precision);
    if (rc) return rc;
    rc = gf_coulomb_finish(ctx, src_precision);
    if (rc) return rc;
    if (dst_precision != src_precision && ctx->pending[dst_precision]) {
        // the destination field is overwritten: its own outstanding update has nothing left to act on.  If its G is
        // the transformation asked for, it has to be used as it stands, so only the flag is dropped.
        ctx->pending[dst_precision] = 0;
    }
    cudaError_t e = launch_apply_transform(g_precision, src_precision, dst_precision, ctx->recon, ctx->gtrans[g_precision],
                                           ctx->links[src_precision], ctx->links[dst_precision], ctx->G, 0, 4, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "gf_apply_transform");
    ctx->launches += 1;
    return GF_OK;
}

// ------------------------------------------------------------------- Coulomb specialisation
extern "C" int gf_set_coulomb_mode(gf_ctx* ctx, int defer_temporal, int freeze_slices)
{
    DeviceGuard guard(ctx);
    if (!ctx) return GF_EINVAL;
    if ((defer_temporal != 0 && defer_temporal != 1) || (freeze_slices != 0 && freeze_slices != 1))
        return fail(ctx, GF_EINVAL, "defer_temporal and freeze_slices must be 0 or 1");
    if (ctx->slab_n > 1 && defer_temporal) return fail(ctx, GF_ESTATE, "deferred temporal links are not available on slabs");
    if (ctx->gauge != GF_COULOMB && (defer_temporal || freeze_slices))
        return fail(ctx, GF_EINVAL, "deferred temporal links and slice freezing exist in Coulomb gauge only");
    if (!defer_temporal) {
        for (int prec = 0; prec < 2; ++prec) {
            int rc = gf_coulomb_finish(ctx, prec);
            if (rc) return rc;
        }
    }
    ctx->defer_temporal = defer_temporal;
    ctx->freeze_slices = freeze_slices;
    return GF_OK;
}

// Turns ctx->host_mask into the ascending list of active slices and uploads it; the copy is ordered on the stream
// between the sweeps.  The callers have drained the stream, so the pinned staging copy is not in flight.
static int upload_mask(gf_ctx* ctx)
{
    int n = 0;
    for (int t = 0; t < ctx->dims[0]; ++t)
        if (ctx->host_mask[t]) ctx->host_list[n++] = (uint16_t)t;
    ctx->n_active = n;
    if (n == 0) return GF_OK;
    cudaError_t e = cudaMemcpyAsync(ctx->dev_list, ctx->host_list, (size_t)n * sizeof(uint16_t), cudaMemcpyHostToDevice, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "slice mask copy");
    return GF_OK;
}

extern "C" int gf_set_slice_mask(gf_ctx* ctx, const uint8_t* host_active)
{
    DeviceGuard guard(ctx);
    if (!ctx) return GF_EINVAL;
    if (ctx->gauge != GF_COULOMB && host_active) return fail(ctx, GF_EINVAL, "slice masks exist in Coulomb gauge only");
    if (!host_active) {
        ctx->mask_on = 0;
        return GF_OK;
    }
    // the pinned staging copy may still be in flight from an earlier call
    cudaError_t e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "gf_set_slice_mask");
    for (int t = 0; t < ctx->dims[0]; ++t) ctx->host_mask[t] = host_active[t] ? 1 : 0;
    ctx->mask_on = 1;
    return upload_mask(ctx);
}

extern "C" int gf_coulomb_finish(gf_ctx* ctx, int precision)
{
    DeviceGuard guard(ctx);
    if (!ctx) return GF_EINVAL;
    if (precision != GF_F32 && precision != GF_F64) return fail(ctx, GF_EINVAL, "precision must be GF_F32 or GF_F64");
    if (!ctx->pending[precision]) return GF_OK;
    if (!ctx->gtrans[precision] || !ctx->links[precision])
        return fail(ctx, GF_ESTATE, "deferred temporal update pending but the transformation buffer was detached");
    // U_0(x) <- G(x) U_0(x) G(x+0)^dagger (eq. 3): the spatial links already carry G
    cudaError_t e = launch_apply_transform(precision, precision, precision, ctx->recon, ctx->gtrans[precision],
                                           ctx->links[precision], ctx->links[precision], ctx->G, 0, 1, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "gf_coulomb_finish");
    ctx->launches += 1;
    ctx->pending[precision] = 0;
    return GF_OK;
}

static int slices_to_host(gf_ctx* ctx, const char* what)
{
    ctx->launches += 2;
    return sync_and_check(ctx, what);
}

extern "C" int gf_plaquette(gf_ctx* ctx, int precision, double* host_out)
{
    DeviceGuard guard(ctx);
    int rc = check_prec(ctx, precision);
    if (rc) return rc;
    rc = gf_coulomb_finish(ctx, precision);
    if (rc) return rc;
    if (!host_out) return fail(ctx, GF_EINVAL, "null output");
    GF_SLAB_BEGIN(ctx);
    cudaError_t e = launch_plaquette(precision, ctx->recon, ctx->links[precision], ctx->next_links[precision], ctx->G, ctx->mg,
                                     ctx->partials, lattice_tail(ctx, 1.0 / (6.0 * 3.0 * (double)ctx->V * ctx->slab_n)), ctx->slice_out,
                                     ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "gf_plaquette launch");
    GF_SLAB_END(ctx);
    rc = slices_to_host(ctx, "gf_plaquette copy");
    if (rc) return rc;
    *host_out = ctx->host_pinned[0];
    return GF_OK;
}

extern "C" int gf_unitarity(gf_ctx* ctx, int precision, double* host_out2)
{
    DeviceGuard guard(ctx);
    int rc = check_prec(ctx, precision);
    if (rc) return rc;
    rc = gf_coulomb_finish(ctx, precision);
    if (rc) return rc;
    if (!host_out2) return fail(ctx, GF_EINVAL, "null output");
    GF_SLAB_BEGIN(ctx);
    cudaError_t e = launch_unitarity(precision, ctx->recon, ctx->links[precision], ctx->G, ctx->mg, ctx->partials, lattice_tail(ctx, 1.0),
                                     ctx->slice_out, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "gf_unitarity launch");
    GF_SLAB_END(ctx);
    rc = slices_to_host(ctx, "gf_unitarity copy");
    if (rc) return rc;
    host_out2[0] = ctx->host_pinned[0];
    host_out2[1] = ctx->host_pinned[1];
    return GF_OK;
}

extern "C" int gf_set_tuning(gf_ctx* ctx, int precision, int lanes_per_site, int block_threads)
{
    DeviceGuard guard(ctx);
    if (!ctx) return GF_EINVAL;
    if (precision != GF_F32 && precision != GF_F64) return fail(ctx, GF_EINVAL, "precision must be GF_F32 or GF_F64");
    if (!sweep_config_valid(lanes_per_site ? lanes_per_site : 1, block_threads ? block_threads : 64))
        return fail(ctx, GF_EINVAL, "lanes must be 0,1,2,4 and block 0, 64, 128 or 256");
    ctx->lanes[precision] = lanes_per_site;
    ctx->block[precision] = block_threads;
    return GF_OK;
}

extern "C" int gf_set_mixed_stall(gf_ctx* ctx, double ratio)
{
    if (!ctx) return GF_EINVAL;
    if (!(ratio >= 0.0 && ratio <= 1.0)) return fail(ctx, GF_EINVAL, "the stall ratio must be in [0, 1]");
    ctx->stall = ratio;
    return GF_OK;
}

extern "C" int gf_set_mixed_handoff(gf_ctx* ctx, double theta_handoff)
{
    DeviceGuard guard(ctx);
    if (!ctx) return GF_EINVAL;
    if (!(theta_handoff > 0.0)) return fail(ctx, GF_EINVAL, "the hand-off theta must be positive");
    ctx->handoff = theta_handoff;
    return GF_OK;
}

extern "C" int gf_set_reunitarize_every(gf_ctx* ctx, int iterations)
{
    if (!ctx) return GF_EINVAL;
    if (iterations < 0) return fail(ctx, GF_EINVAL, "negative re-projection interval");
    ctx->reunit_every = iterations;
    return GF_OK;
}

extern "C" int gf_set_fix_runahead(gf_ctx* ctx, int blocks)
{
    if (!ctx) return GF_EINVAL;
    if (blocks < 0 || blocks > kRunAhead) return fail(ctx, GF_EINVAL, "run-ahead must be 0..%d evaluation blocks", kRunAhead);
    ctx->runahead = blocks;
    return GF_OK;
}

extern "C" int gf_set_traversal(gf_ctx* ctx, int zigzag)
{
    DeviceGuard guard(ctx);
    if (!ctx) return GF_EINVAL;
    if (zigzag != 0 && zigzag != 1) return fail(ctx, GF_EINVAL, "traversal must be 0 (forward) or 1 (zigzag)");
    ctx->zigzag = zigzag;
    return GF_OK;
}

extern "C" int gf_set_solver_precision(gf_ctx* ctx, int solver_precision)
{
    DeviceGuard guard(ctx);
    if (!ctx) return GF_EINVAL;
    if (solver_precision != GF_F32 && solver_precision != GF_F64 && solver_precision != GF_SOLVER_AUTO)
        return fail(ctx, GF_EINVAL, "solver precision must be GF_F32, GF_F64 or GF_SOLVER_AUTO");
    ctx->solver_mode = solver_precision;
    return GF_OK;
}

extern "C" int gf_debug_philox(gf_ctx* ctx, int n, const uint32_t* dev_counters, const uint32_t* dev_keys, uint32_t* dev_out)
{
    DeviceGuard guard(ctx);
    if (!ctx) return GF_EINVAL;
    if (n < 0 || !dev_counters || !dev_keys || !dev_out) return fail(ctx, GF_EINVAL, "bad arguments");
    if (n == 0) return GF_OK;
    cudaError_t e = launch_philox(n, dev_counters, dev_keys, dev_out, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "gf_debug_philox");
    ctx->launches += 1;
    return GF_OK;
}

extern "C" int gf_launch_count(const gf_ctx* ctx, uint64_t* count_out)
{
    if (!ctx || !count_out) return GF_EINVAL;
    *count_out = ctx->launches;
    return GF_OK;
}
