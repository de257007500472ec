// gf_static.cu -- gf_measure_static: F and theta of a link field for callers that may not allocate.
//
// Everything else in this library needs a gf_ctx, and gf_init_lattice allocates: a context on the heap, pinned host
// memory for the results (cudaMallocHost), events -- and it wants a workspace buffer the caller had to cudaMalloc.
// That rules it out for code that runs where allocation is off limits: a convergence monitor hooked into someone
// else's update loop after that application has handed the whole GPU to its pool allocator (a raw cudaMalloc then
// fails, and the pool is not ours to ask); a job whose memory budget is fixed at start-up and audited; a latency-bound
// loop that cannot take the device-wide synchronisation cudaMalloc / cudaMallocHost / cudaFree imply.  For those
// callers this file offers one call that takes the link field and an output pointer and nothing else.
//
// The reduction needs scratch between its two kernels (per-block partial sums, per-slice sums, the counter that
// elects the last block).  Here that scratch is the file-scope array g_scratch below: it is part of the library's
// device image, so every GPU on which the library gets loaded holds kStaticScratchBytes (a little over 1 MiB) of it
// from then until the process exits, whether or not this entry point is ever called.  That fixed size is the limit of
// the call: lattices whose reduction needs more than GF_STATIC_MAX_BLOCKS partial sums are refused (see include/gf.h).
//
// The kernels are the ones gf_measure runs (measure_kernel, reduce_slices_kernel in gf_aux.cu, reached through
// launch_measure); only where their scratch lives differs, so the results are bitwise those of gf_measure.
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "../../include/gf.h"
#include "gf_internal.h"

using namespace gf;

namespace {

// layout of the scratch: [counter word, padded to 256 B][slice_tmp: 2 doubles per time slice, N_t <= 4096][partials]
constexpr size_t kMaxNtStatic = 4096;
constexpr size_t kCounterBytes = 256;
constexpr size_t kSliceTmpBytes = 2 * kMaxNtStatic * sizeof(double);
constexpr size_t kPartialBytes = (size_t)GF_STATIC_MAX_BLOCKS * 2 * sizeof(double);
constexpr size_t kStaticScratchBytes = kCounterBytes + kSliceTmpBytes + kPartialBytes;      // 1 114 368 bytes
constexpr int kMaxDevices = 64;

}  // namespace

// In HOST code the name g_scratch is only a handle for the runtime (a host-side shadow variable): its host address is
// not a device address, and a kernel handed &g_scratch[0] from host code would fault -- or, on systems where the GPU
// can reach host memory, quietly reduce into the wrong memory.  Host code must ask the runtime where the array lives
// on the current device (scratch_for_current_device below); device code in this file may name it directly.
static __device__ __align__(256) unsigned char g_scratch[kStaticScratchBytes];

namespace {

// The one word of the scratch that has to be zero when a reduction starts: the count of finished blocks of the last
// stage.  reduce_slices_kernel leaves it at zero itself, but the array is shared by every call and keeps what the
// last one left -- after a call that was cut short (a faulting launch elsewhere on the stream, a reset of the
// caller's making) it need not be.  Partial sums and slice sums are written in full before they are read.
__global__ void static_scratch_reset_kernel()
{
    if (threadIdx.x == 0) *reinterpret_cast<uint32_t*>(g_scratch) = 0u;
}

std::mutex g_setup_lock;
unsigned char* g_scratch_dev[kMaxDevices];      // device address of g_scratch per CUDA device, nullptr = not set up yet

int static_fail(char* host_err, size_t host_err_len, int code, const char* fmt, ...)
{
    if (host_err && host_err_len) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(host_err, host_err_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

// Set-up, once per device, with that device current: the device address of g_scratch.  No allocation: the array came
// with the module.  (The very first CUDA call of a process on a device creates the primary context and loads the
// module; that is the runtime's doing and happens for any entry point of the library.)
int scratch_for_current_device(unsigned char** out, char* host_err, size_t host_err_len)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return static_fail(host_err, host_err_len, GF_ECUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices)
        return static_fail(host_err, host_err_len, GF_ECUDA, "device ordinal %d is beyond the %d this entry point keeps a scratch address for", dev, kMaxDevices);
    std::lock_guard<std::mutex> hold(g_setup_lock);
    if (!g_scratch_dev[dev]) {
        int major = 0;
        e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
        if (e != cudaSuccess) return static_fail(host_err, host_err_len, GF_ECUDA, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
        if (major != 10) return static_fail(host_err, host_err_len, GF_ECUDA, "device %d is sm_%dx; the library is built for sm_100a only", dev, major);
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_scratch);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return static_fail(host_err, host_err_len, GF_ECUDA, "cudaGetSymbolAddress(static scratch) on device %d: %s", dev, cudaGetErrorString(e));
        }
        g_scratch_dev[dev] = static_cast<unsigned char*>(p);
    }
    *out = g_scratch_dev[dev];
    return GF_OK;
}

}  // namespace

extern "C" int gf_measure_static(const int dims[4], int gauge, int precision, int recon, const void* dev_links,
                                 double* dev_out, void* cuda_stream, char* host_err, size_t host_err_len)
{
    if (host_err && host_err_len) host_err[0] = '\0';
    if (!dims) return static_fail(host_err, host_err_len, GF_EINVAL, "dims is NULL");
    uint64_t V = 1;
    for (int i = 0; i < 4; ++i) {
        if (dims[i] < 2 || (dims[i] & 1))
            return static_fail(host_err, host_err_len, GF_EINVAL, "dims[%d] = %d: every extent must be even and >= 2", i, dims[i]);
        V *= (uint64_t)dims[i];
    }
    if ((size_t)dims[0] > kMaxNtStatic || V >= (uint64_t(1) << 32))
        return static_fail(host_err, host_err_len, GF_EINVAL, "lattice too large for the library (N_t <= 4096, fewer than 2^32 sites)");
    if (gauge != GF_LANDAU && gauge != GF_COULOMB) return static_fail(host_err, host_err_len, GF_EINVAL, "gauge must be GF_LANDAU or GF_COULOMB");
    if (precision != GF_F32 && precision != GF_F64) return static_fail(host_err, host_err_len, GF_EINVAL, "precision must be GF_F32 or GF_F64");
    if (recon != GF_RECON18 && recon != GF_RECON12) return static_fail(host_err, host_err_len, GF_EINVAL, "recon must be GF_RECON18 or GF_RECON12");
    if (!dev_links || !dev_out) return static_fail(host_err, host_err_len, GF_EINVAL, "dev_links and dev_out must not be NULL");
    if ((uintptr_t)dev_links & 15u) return static_fail(host_err, host_err_len, GF_EINVAL, "dev_links must be 16-byte aligned");
    if ((uintptr_t)dev_out & 7u) return static_fail(host_err, host_err_len, GF_EINVAL, "dev_out must be 8-byte aligned");

    const MeasureGrid mg = make_measure_grid(dims);
    const uint64_t blocks = (uint64_t)dims[0] * 2u * mg.bpp;
    if (blocks > (uint64_t)GF_STATIC_MAX_BLOCKS)
        return static_fail(host_err, host_err_len, GF_EINVAL,
                           "lattice %dx%dx%dx%d needs %llu partial sums (N_t * 2 * ceil(N_x N_y N_z / %u)); the static scratch of "
                           "gf_measure_static holds GF_STATIC_MAX_BLOCKS = %d: use gf_measure with a workspace of your own",
                           dims[0], dims[1], dims[2], dims[3], (unsigned long long)blocks, 2u * kMeasureBlockThreads, (int)GF_STATIC_MAX_BLOCKS);

    unsigned char* scratch = nullptr;
    int rc = scratch_for_current_device(&scratch, host_err, host_err_len);
    if (rc) return rc;

    ReduceTail tail;
    tail.counter = reinterpret_cast<uint32_t*>(scratch);
    tail.slice_tmp = reinterpret_cast<double*>(scratch + kCounterBytes);
    double* partials = reinterpret_cast<double*>(scratch + kCounterBytes + kSliceTmpBytes);
    tail.stop = nullptr;
    tail.target = 0.0;
    tail.stall = 0.0;
    tail.prev = nullptr;
    // normalisations of PAPER.md:39 (eq. 2) and :52 (eq. 5), as gf_measure applies them
    if (gauge == GF_COULOMB) {
        const double Vs = (double)(V / (uint64_t)dims[0]);
        tail.combine = 0;
        tail.scale0 = 1.0 / (3.0 * 3.0 * Vs);
        tail.scale1 = 1.0 / (3.0 * Vs);
    } else {
        tail.combine = 1;
        tail.scale0 = 1.0 / (3.0 * 4.0 * (double)V);
        tail.scale1 = 1.0 / (3.0 * (double)V);
    }

    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    static_scratch_reset_kernel<<<1, 32, 0, st>>>();
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return static_fail(host_err, host_err_len, GF_ECUDA, "scratch reset launch: %s", cudaGetErrorString(e));
    e = launch_measure(precision, recon, dev_links, nullptr, make_geom(dims), gauge == GF_COULOMB ? 1 : 0, mg, partials, tail, dev_out, st);
    if (e != cudaSuccess) return static_fail(host_err, host_err_len, GF_ECUDA, "measure launch: %s", cudaGetErrorString(e));
    return GF_OK;
}
