// gf_aux.cu -- everything around the sweep: the F / theta reduction,
// diagnostics (plaquette, unitarity), layout conversion (pack / unpack / cast) and the Philox
// known-answer kernel.  All of it is HBM bound and off the inner loop; the reductions use a
// fixed order (warp shuffle -> shared memory -> per-block partials -> one block per time slice),
// no floating-point atomics.
#include "gf_internal.h"

namespace gf {

// ------------------------------------------------------------------------------ reductions
struct OpSum {
    __device__ static double apply(double a, double b) { return a + b; }
};
struct OpMax {   // of non-negative values, so 0 is neutral for both
    __device__ static double apply(double a, double b) { return fmax(a, b); }
};

template <typename Op>
__device__ __forceinline__ double warp_reduce(double v)
{
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v = Op::apply(v, __shfl_xor_sync(0xffffffffu, v, off));
    return v;
}

// Reduces two values per thread over the block; thread 0 writes them to out[0], out[1].
template <typename Op>
__device__ __forceinline__ void block_reduce2(double a, double b, double* out)
{
    __shared__ double sh[2][32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    a = warp_reduce<Op>(a);
    b = warp_reduce<Op>(b);
    if (lane == 0) {
        sh[0][w] = a;
        sh[1][w] = b;
    }
    __syncthreads();
    if (w == 0) {
        a = lane < nw ? sh[0][lane] : 0.0;
        b = lane < nw ? sh[1][lane] : 0.0;
        a = warp_reduce<Op>(a);
        b = warp_reduce<Op>(b);
        if (lane == 0) {
            out[0] = a;
            out[1] = b;
        }
    }
}

// a9, last stage.  One block per time slice combines that slice's per-block partials in a fixed order and
// scales them (the normalisations of PAPER.md:39 and :52).  COMBINE = 0 (Coulomb gauge: one value per
// time slice): out[2t], out[2t+1].  COMBINE = 1 (values of the whole lattice): the slice values go to
// slice_tmp and the block that finishes last -- known from a counter it resets -- folds all N_t of
// them, again in a fixed order, into out[0], out[1].  `out` may be mapped pinned host memory: the host
// reads finished results and does no arithmetic of the method.

// The stopping decision of the run-ahead fix loop, taken by the last thread of the last reduction stage on the value
// the host will read from pinned memory, with the comparisons the host makes (gf_api.cu, fix_phase_runahead):
// theta below the target, or -- fp32 phase of the mixed-precision runs, tail.stall > 0 -- theta not below stall x the
// previous evaluation's (>=: a bit-identical plateau at the rounding floor counts as stalled).
__device__ __forceinline__ void decide_stop(const ReduceTail& tail, double th)
{
    bool stop = th < tail.target;
    if (tail.stall > 0.0) {
        const double prev = *tail.prev;
        if (prev > 0.0 && th >= tail.stall * prev) stop = true;
        *tail.prev = th;
    }
    if (stop) *tail.stop = 1u;
}

template <typename Op>
__global__ void reduce_slices_kernel(const double* __restrict__ partials, uint32_t per_slice, const ReduceTail tail,
                                     double* __restrict__ out, const uint16_t* __restrict__ slice_list)
{
    __shared__ double res[2];
    __shared__ uint32_t last;
    // block -> time slice; with a list (per-slice results only, tail.combine == 0) the listed slices
    const uint32_t slice = slice_list ? slice_list[blockIdx.x] : blockIdx.x;
    const double* p = partials + (size_t)slice * per_slice * 2;
    double a = 0.0, b = 0.0;
    for (uint32_t i = threadIdx.x; i < per_slice; i += blockDim.x) {
        a = Op::apply(a, p[2 * i]);
        b = Op::apply(b, p[2 * i + 1]);
    }
    block_reduce2<Op>(a, b, res);
    if (!tail.combine) {
        if (threadIdx.x == 0) {
            out[2 * slice] = res[0] * tail.scale0;
            out[2 * slice + 1] = res[1] * tail.scale1;
        }
        if (tail.stop == nullptr) return;
        // run-ahead fix loop, Coulomb gauge: the block that finishes last decides max_t theta_t < target
        if (threadIdx.x == 0) {
            tail.slice_tmp[blockIdx.x] = res[1] * tail.scale1;
            __threadfence();
            last = atomicAdd(tail.counter, 1u) == gridDim.x - 1u ? 1u : 0u;
        }
        __syncthreads();
        if (!last) return;
        __threadfence();
        a = b = 0.0;
        for (uint32_t t = threadIdx.x; t < gridDim.x; t += blockDim.x) a = fmax(a, __ldcg(tail.slice_tmp + t));
        __syncthreads();
        block_reduce2<OpMax>(a, b, res);
        if (threadIdx.x == 0) {
            decide_stop(tail, res[0]);
            *tail.counter = 0u;
        }
        return;
    }
    if (threadIdx.x == 0) {
        tail.slice_tmp[2 * blockIdx.x] = res[0];
        tail.slice_tmp[2 * blockIdx.x + 1] = res[1];
        __threadfence();
        last = atomicAdd(tail.counter, 1u) == gridDim.x - 1u ? 1u : 0u;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    a = b = 0.0;
    for (uint32_t t = threadIdx.x; t < gridDim.x; t += blockDim.x) {
        a = Op::apply(a, __ldcg(tail.slice_tmp + 2 * t));
        b = Op::apply(b, __ldcg(tail.slice_tmp + 2 * t + 1));
    }
    __syncthreads();                                    // block_reduce2's scratch is reused
    block_reduce2<Op>(a, b, res);
    if (threadIdx.x == 0) {
        const double th = res[1] * tail.scale1;
        out[0] = res[0] * tail.scale0;
        out[1] = th;
        if (tail.stop != nullptr) decide_stop(tail, th);
        *tail.counter = 0u;
    }
}

// blockIdx.y -> time slice: all of them, or the listed ones (Coulomb slice freezing: frozen slices keep their results)
__device__ __forceinline__ uint32_t measure_slice(const MeasureGrid& mg)
{
    return mg.slice_list ? mg.slice_list[blockIdx.y] : blockIdx.y;
}

// thread -> (slice t, parity, site) of the measurement grids: blockIdx.y -> t, blockIdx.x = 2*chunk + parity
__device__ __forceinline__ bool measure_site(const Geom& G, const MeasureGrid& mg, uint32_t& parity, Site& s)
{
    parity = blockIdx.x & 1u;
    const uint32_t i = (blockIdx.x >> 1) * blockDim.x + threadIdx.x;
    const bool live = i < mg.Sh;
    const uint32_t h = measure_slice(mg) * mg.Sh + (live ? i : mg.Sh - 1u);
    s = decode_site(G, h, parity);
    return live;
}

__device__ __forceinline__ size_t partial_slot(const MeasureGrid& mg)
{
    return ((size_t)measure_slice(mg) * (2u * mg.bpp) + blockIdx.x) * 2;
}

// a7 + a8: per-block partial sums of  sum_mu Re tr U_mu(x)  and  tr[Delta(x) Delta(x)^dagger].
// Delta(x) = sum_mu (A_mu(x) - A_mu(x-mu)) with A the traceless anti-Hermitian part of U
// (eq. 4); as A is linear in U, Delta = traceless[(M - M^dagger)/(2i)] with
// M = sum_mu (U_mu(x) - U_mu(x-mu)).  Accumulation in fp64 whatever the storage precision.
template <typename T, int RECON>
__global__ void measure_kernel(const T* __restrict__ links, const T* __restrict__ prev_links, const Geom G, const int mu0,
                               const MeasureGrid mg, double* __restrict__ partials)
{
    uint32_t parity;
    Site s;
    const bool live = measure_site(G, mg, parity, s);
    double M[18];
#pragma unroll
    for (int k = 0; k < 18; ++k) M[k] = 0.0;
    double F = 0.0;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        if (mu < mu0) continue;
        T Uf[18], Ub[18];
        load_link<RECON>(links + block_offset<T>(parity, mu, RECON, G), s.h, Uf);
        const T* back = (mu == 0 && s.c[0] == 0) ? prev_links : links;     // slab below for the first local slice
        load_link<RECON>(back + block_offset<T>(parity ^ 1u, mu, RECON, G), backward_index(G, s, mu), Ub);
        if (RECON == 12) {
            reconstruct_row2(Uf);
            reconstruct_row2(Ub);
        }
        F += (double)Uf[0] + (double)Uf[8] + (double)Uf[16];
#pragma unroll
        for (int k = 0; k < 18; ++k) M[k] += (double)Uf[k] - (double)Ub[k];
    }
    // diagonal of (M - M^dagger)/(2i) is Im M_aa; off-diagonal |.|^2 = |M_ab - conj(M_ba)|^2 / 4
    const double tr3 = (GF_IM(M, 0, 0) + GF_IM(M, 1, 1) + GF_IM(M, 2, 2)) * (1.0 / 3.0);
    double th = 0.0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double d = GF_IM(M, a, a) - tr3;
        th += d * d;
    }
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = a + 1; b < 3; ++b) {
            const double dr = GF_RE(M, a, b) - GF_RE(M, b, a), di = GF_IM(M, a, b) + GF_IM(M, b, a);
            th += 0.5 * (dr * dr + di * di);
        }
    if (!live) {
        F = 0.0;
        th = 0.0;
    }
    block_reduce2<OpSum>(F, th, partials + partial_slot(mg));
}

template <typename T, int RECON>
__device__ __forceinline__ void load_full_d(const T* links, const Geom& G, uint32_t parity, int mu, uint32_t h, double (&m)[18])
{
    T u[18];
    load_link<RECON>(links + block_offset<T>(parity, mu, RECON, G), h, u);
    if (RECON == 12) reconstruct_row2(u);
#pragma unroll
    for (int k = 0; k < 18; ++k) m[k] = (double)u[k];
}

__device__ __forceinline__ void mul_full(const double (&A)[18], const double (&B)[18], double (&C)[18], bool dagger_b)
{
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            double re = 0.0, im = 0.0;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const double br = dagger_b ? GF_RE(B, b, k) : GF_RE(B, k, b);
                const double bi = dagger_b ? -GF_IM(B, b, k) : GF_IM(B, k, b);
                re += GF_RE(A, a, k) * br - GF_IM(A, a, k) * bi;
                im += GF_RE(A, a, k) * bi + GF_IM(A, a, k) * br;
            }
            GF_RE(C, a, b) = re;
            GF_IM(C, a, b) = im;
        }
}

// sum_{mu<nu} Re tr[U_mu(x) U_nu(x+mu) U_mu(x+nu)^dagger U_nu(x)^dagger]   (diagnostic)
template <typename T, int RECON>
__global__ void plaquette_kernel(const T* __restrict__ links, const T* __restrict__ next_links, const Geom G,
                                 const MeasureGrid mg, double* __restrict__ partials)
{
    uint32_t parity;
    Site s;
    const bool live = measure_site(G, mg, parity, s);
    double sum = 0.0;
    for (int mu = 0; mu < 4; ++mu)
        for (int nu = mu + 1; nu < 4; ++nu) {
            double A[18], B[18], C[18], D[18];
            load_full_d<T, RECON>(links, G, parity, mu, s.h, A);
            // x + mu_hat leaves the slab through its last time slice only for mu = 0
            load_full_d<T, RECON>((mu == 0 && s.c[0] + 1u == G.nt) ? next_links : links, G, parity ^ 1u, nu, forward_index(G, s, mu), B);
            mul_full(A, B, C, false);
            load_full_d<T, RECON>(links, G, parity ^ 1u, mu, forward_index(G, s, nu), A);
            mul_full(C, A, D, true);
            load_full_d<T, RECON>(links, G, parity, nu, s.h, B);
            // Re tr[D B^dagger] = sum_ab Re(D_ab conj(B_ab))
#pragma unroll
            for (int k = 0; k < 18; ++k) sum += D[k] * B[k];
        }
    if (!live) sum = 0.0;
    block_reduce2<OpSum>(sum, 0.0, partials + partial_slot(mg));
}

// max |U U^dagger - 1| entry and max |det U - 1| over the four links stored at each site
template <typename T, int RECON>
__global__ void unitarity_kernel(const T* __restrict__ links, const Geom G, const MeasureGrid mg,
                                 double* __restrict__ partials)
{
    uint32_t parity;
    Site s;
    measure_site(G, mg, parity, s);    // a clamped duplicate site does not change a maximum
    double dmax = 0.0, detmax = 0.0;
    for (int mu = 0; mu < 4; ++mu) {
        double U[18], P[18];
        load_full_d<T, RECON>(links, G, parity, mu, s.h, U);
        mul_full(U, U, P, true);
        P[0] -= 1.0;
        P[8] -= 1.0;
        P[16] -= 1.0;
#pragma unroll
        for (int k = 0; k < 9; ++k) dmax = fmax(dmax, sqrt(P[2 * k] * P[2 * k] + P[2 * k + 1] * P[2 * k + 1]));
        // det U = row0 . (row1 x row2)
        double dr = 0.0, di = 0.0;
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const int b1 = (b + 1) % 3, b2 = (b + 2) % 3;
            const double cr = GF_RE(U, 1, b1) * GF_RE(U, 2, b2) - GF_IM(U, 1, b1) * GF_IM(U, 2, b2)
                            - GF_RE(U, 1, b2) * GF_RE(U, 2, b1) + GF_IM(U, 1, b2) * GF_IM(U, 2, b1);
            const double ci = GF_RE(U, 1, b1) * GF_IM(U, 2, b2) + GF_IM(U, 1, b1) * GF_RE(U, 2, b2)
                            - GF_RE(U, 1, b2) * GF_IM(U, 2, b1) - GF_IM(U, 1, b2) * GF_RE(U, 2, b1);
            dr += GF_RE(U, 0, b) * cr - GF_IM(U, 0, b) * ci;
            di += GF_RE(U, 0, b) * ci + GF_IM(U, 0, b) * cr;
        }
        detmax = fmax(detmax, sqrt((dr - 1.0) * (dr - 1.0) + di * di));
    }
    block_reduce2<OpMax>(dmax, detmax, partials + partial_slot(mg));
}

template <template <typename, int> class Launcher, typename... Args>
static cudaError_t dispatch(int precision, int recon, Args... args)
{
    if (precision == PREC_F64)
        return recon == 12 ? Launcher<double, 12>::run(args...) : Launcher<double, 18>::run(args...);
    return recon == 12 ? Launcher<float, 12>::run(args...) : Launcher<float, 18>::run(args...);
}

static dim3 measure_dims(const Geom& G, const MeasureGrid& mg) { return dim3(2u * mg.bpp, mg.slice_list ? mg.n_listed : G.nt, 1); }

template <typename T, int RECON> struct MeasureLauncher {
    static cudaError_t run(const void* links, const void* prev_links, const Geom& G, int mu0, const MeasureGrid& mg, double* partials,
                           const ReduceTail& tail, double* slice_out, cudaStream_t st)
    {
        uniform_carveout(measure_kernel<T, RECON>);
        measure_kernel<T, RECON><<<measure_dims(G, mg), mg.block, 0, st>>>(static_cast<const T*>(links),
                                                                           static_cast<const T*>(prev_links ? prev_links : links), G, mu0, mg, partials);
        uniform_carveout(reduce_slices_kernel<OpSum>);
        reduce_slices_kernel<OpSum><<<measure_dims(G, mg).y, 256, 0, st>>>(partials, 2u * mg.bpp, tail, slice_out, mg.slice_list);
        return cudaGetLastError();
    }
};

template <typename T, int RECON> struct PlaquetteLauncher {
    static cudaError_t run(const void* links, const void* next_links, const Geom& G, const MeasureGrid& mg, double* partials,
                           const ReduceTail& tail, double* slice_out, cudaStream_t st)
    {
        uniform_carveout(plaquette_kernel<T, RECON>);
        plaquette_kernel<T, RECON><<<measure_dims(G, mg), mg.block, 0, st>>>(static_cast<const T*>(links),
                                                                             static_cast<const T*>(next_links ? next_links : links), G, mg, partials);
        uniform_carveout(reduce_slices_kernel<OpSum>);
        reduce_slices_kernel<OpSum><<<measure_dims(G, mg).y, 256, 0, st>>>(partials, 2u * mg.bpp, tail, slice_out, mg.slice_list);
        return cudaGetLastError();
    }
};

template <typename T, int RECON> struct UnitarityLauncher {
    static cudaError_t run(const void* links, const Geom& G, const MeasureGrid& mg, double* partials,
                           const ReduceTail& tail, double* slice_out, cudaStream_t st)
    {
        uniform_carveout(unitarity_kernel<T, RECON>);
        unitarity_kernel<T, RECON><<<measure_dims(G, mg), mg.block, 0, st>>>(static_cast<const T*>(links), G, mg, partials);
        uniform_carveout(reduce_slices_kernel<OpMax>);
        reduce_slices_kernel<OpMax><<<measure_dims(G, mg).y, 256, 0, st>>>(partials, 2u * mg.bpp, tail, slice_out, mg.slice_list);
        return cudaGetLastError();
    }
};

cudaError_t launch_measure(int precision, int recon, const void* links, const void* prev_links, const Geom& G, int mu0,
                           const MeasureGrid& mg, double* partials, const ReduceTail& tail, double* slice_out, cudaStream_t st)
{
    return dispatch<MeasureLauncher>(precision, recon, links, prev_links, G, mu0, mg, partials, tail, slice_out, st);
}

cudaError_t launch_plaquette(int precision, int recon, const void* links, const void* next_links, const Geom& G,
                             const MeasureGrid& mg, double* partials, const ReduceTail& tail, double* slice_out, cudaStream_t st)
{
    return dispatch<PlaquetteLauncher>(precision, recon, links, next_links, G, mg, partials, tail, slice_out, st);
}

cudaError_t launch_unitarity(int precision, int recon, const void* links, const Geom& G,
                             const MeasureGrid& mg, double* partials, const ReduceTail& tail, double* slice_out, cudaStream_t st)
{
    return dispatch<UnitarityLauncher>(precision, recon, links, G, mg, partials, tail, slice_out, st);
}

// ---------------------------------------------------------------------- pack / unpack / cast
// a11: canonical AoS (site s, mu, 3x3 row-major complex) <-> the private tiled layout, transposed through a small
// shared-memory tile so that BOTH sides move whole 16-byte vectors to consecutive addresses.  A block takes a
// segment of PACK_TH consecutive half-indices of one x-row: with both parities that is 2 * PACK_TH consecutive
// canonical sites (x = 2 xh + xodd, the two parities interleave along x), i.e. one contiguous canonical range of
// 2 * PACK_TH * 72 reals = 9216 bytes in fp64.  One thread per link does the private-layout side (load_link /
// store_link: 16-byte chunks, consecutive lanes consecutive sites; reconstruction of row 2 for 12-real storage), all
// threads stream the canonical side.  64 threads and at most 9 KB of static shared memory per block: such blocks
// co-reside with the register-bound sweep blocks of other lattices in flight (the round-1 transpose, with large
// dynamic tiles, did not: it was 3.6x faster alone and slowed the pipelined end-to-end step).
constexpr uint32_t PACK_TH = 8;                       // half-indices per segment
constexpr uint32_t PACK_THREADS = 2 * 4 * PACK_TH;    // one thread per (parity, mu, site) link

struct PackSegment {
    uint32_t h0, len;       // first half-index and number of sites (<= PACK_TH; the last segment of a row may be short)
    uint32_t xodd0;         // x & 1 of the parity-0 sites of this row
    size_t site0;           // canonical index of the first site of the range: 2 * h0
};

__device__ __forceinline__ PackSegment pack_segment(const Geom& G, uint32_t segs_per_row)
{
    PackSegment p;
    const uint32_t row = blockIdx.x / segs_per_row, seg = blockIdx.x - row * segs_per_row;
    p.h0 = row * G.nxh + seg * PACK_TH;
    p.len = min(PACK_TH, G.nxh - seg * PACK_TH);
    const Site s = decode_site(G, p.h0, 0u);
    p.xodd0 = s.xodd;
    p.site0 = 2u * (size_t)p.h0;
    return p;
}

template <typename T, int RECON, typename TC>
__global__ void __launch_bounds__(PACK_THREADS) pack_kernel(T* __restrict__ links, const Geom G, const uint32_t segs_per_row,
                                                            const TC* __restrict__ canonical)
{
    __shared__ __align__(16) TC tile[2 * PACK_TH * 72];
    const PackSegment p = pack_segment(G, segs_per_row);
    // canonical -> shared: one contiguous range, 16-byte vectors (72 reals per site: always whole vectors)
    using V = typename Vec16<TC>::type;
    constexpr uint32_t PER = 16u / (uint32_t)sizeof(TC);
    const uint32_t nvec = 2u * p.len * 72u / PER;
    const V* src = reinterpret_cast<const V*>(canonical + p.site0 * 72u);
    for (uint32_t i = threadIdx.x; i < nvec; i += PACK_THREADS) reinterpret_cast<V*>(tile)[i] = src[i];
    __syncthreads();
    // shared -> private layout: thread = (parity, mu, k)
    const uint32_t k = threadIdx.x % PACK_TH, mu = (threadIdx.x / PACK_TH) & 3u, parity = threadIdx.x / (4u * PACK_TH);
    if (k >= p.len) return;
    const uint32_t local = 2u * k + (p.xodd0 ^ parity);          // site of this parity inside the canonical range
    T m[18];
#pragma unroll
    for (int q = 0; q < 18; ++q) m[q] = (T)tile[(local * 4u + mu) * 18u + q];
    store_link<RECON>(links + block_offset<T>(parity, (int)mu, RECON, G), p.h0 + k, m);
}

template <typename T, int RECON, typename TC>
__global__ void __launch_bounds__(PACK_THREADS) unpack_kernel(const T* __restrict__ links, const Geom G, const uint32_t segs_per_row,
                                                              TC* __restrict__ canonical)
{
    __shared__ __align__(16) TC tile[2 * PACK_TH * 72];
    const PackSegment p = pack_segment(G, segs_per_row);
    const uint32_t k = threadIdx.x % PACK_TH, mu = (threadIdx.x / PACK_TH) & 3u, parity = threadIdx.x / (4u * PACK_TH);
    if (k < p.len) {
        const uint32_t local = 2u * k + (p.xodd0 ^ parity);
        T m[18];
        load_link<RECON>(links + block_offset<T>(parity, (int)mu, RECON, G), p.h0 + k, m);
        if (RECON == 12) reconstruct_row2(m);
#pragma unroll
        for (int q = 0; q < 18; ++q) tile[(local * 4u + mu) * 18u + q] = (TC)m[q];
    }
    __syncthreads();
    using V = typename Vec16<TC>::type;
    constexpr uint32_t PER = 16u / (uint32_t)sizeof(TC);
    const uint32_t nvec = 2u * p.len * 72u / PER;
    V* dst = reinterpret_cast<V*>(canonical + p.site0 * 72u);
    for (uint32_t i = threadIdx.x; i < nvec; i += PACK_THREADS) dst[i] = reinterpret_cast<const V*>(tile)[i];
}

// Gram-Schmidt on rows 0 and 1, row 2 = conj(row 0 x row 1)
__device__ __forceinline__ void project_su3(double (&m)[18])
{
    double n0 = 0.0;
#pragma unroll
    for (int k = 0; k < 6; ++k) n0 += m[k] * m[k];
    n0 = 1.0 / sqrt(n0);
#pragma unroll
    for (int k = 0; k < 6; ++k) m[k] *= n0;
    double pr = 0.0, pi = 0.0;                       // conj(row0) . row1
#pragma unroll
    for (int b = 0; b < 3; ++b) {
        pr += GF_RE(m, 0, b) * GF_RE(m, 1, b) + GF_IM(m, 0, b) * GF_IM(m, 1, b);
        pi += GF_RE(m, 0, b) * GF_IM(m, 1, b) - GF_IM(m, 0, b) * GF_RE(m, 1, b);
    }
#pragma unroll
    for (int b = 0; b < 3; ++b) {
        GF_RE(m, 1, b) -= pr * GF_RE(m, 0, b) - pi * GF_IM(m, 0, b);
        GF_IM(m, 1, b) -= pr * GF_IM(m, 0, b) + pi * GF_RE(m, 0, b);
    }
    double n1 = 0.0;
#pragma unroll
    for (int k = 6; k < 12; ++k) n1 += m[k] * m[k];
    n1 = 1.0 / sqrt(n1);
#pragma unroll
    for (int k = 6; k < 12; ++k) m[k] *= n1;
    reconstruct_row2(m);
}

// every (parity, mu, h) link: load as TS, optionally re-project in fp64, store as TD
template <typename TS, typename TD, int RECON>
__global__ void cast_kernel(const TS* src, TD* dst, const Geom G, const int reproject, const uint32_t* stop)   // src may alias dst
{
    const uint32_t h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= G.Vh) return;
    if (stop != nullptr && *stop != 0u) return;      // run-ahead fix loop: enqueued behind the evaluation that met the target
    const uint32_t pm = blockIdx.y;                  // parity*4 + mu
    TS u[18];
    load_link<RECON>(src + (size_t)pm * RECON * padded_vh<TS>(G), h, u);
    double m[18];
#pragma unroll
    for (int k = 0; k < 18; ++k) m[k] = (double)u[k];
    if (reproject) project_su3(m);
    TD o[18];
#pragma unroll
    for (int k = 0; k < 18; ++k) o[k] = (TD)m[k];
    store_link<RECON>(dst + (size_t)pm * RECON * padded_vh<TD>(G), h, o);
}

static uint32_t pack_segments_per_row(const Geom& G) { return (G.nxh + PACK_TH - 1u) / PACK_TH; }

template <typename T, int RECON>
static cudaError_t pack_run(void* links, const Geom& G, const void* canonical, int canonical_is_f64, cudaStream_t st)
{
    const uint32_t spr = pack_segments_per_row(G), grid = G.Vh / G.nxh * spr;
    if (canonical_is_f64) {
        uniform_carveout(pack_kernel<T, RECON, double>);
        pack_kernel<T, RECON, double><<<grid, PACK_THREADS, 0, st>>>(static_cast<T*>(links), G, spr, static_cast<const double*>(canonical));
    } else {
        uniform_carveout(pack_kernel<T, RECON, float>);
        pack_kernel<T, RECON, float><<<grid, PACK_THREADS, 0, st>>>(static_cast<T*>(links), G, spr, static_cast<const float*>(canonical));
    }
    return cudaGetLastError();
}

template <typename T, int RECON>
static cudaError_t unpack_run(const void* links, const Geom& G, void* canonical, int canonical_is_f64, cudaStream_t st)
{
    const uint32_t spr = pack_segments_per_row(G), grid = G.Vh / G.nxh * spr;
    if (canonical_is_f64) {
        uniform_carveout(unpack_kernel<T, RECON, double>);
        unpack_kernel<T, RECON, double><<<grid, PACK_THREADS, 0, st>>>(static_cast<const T*>(links), G, spr, static_cast<double*>(canonical));
    } else {
        uniform_carveout(unpack_kernel<T, RECON, float>);
        unpack_kernel<T, RECON, float><<<grid, PACK_THREADS, 0, st>>>(static_cast<const T*>(links), G, spr, static_cast<float*>(canonical));
    }
    return cudaGetLastError();
}

cudaError_t launch_pack(int precision, int recon, void* links, const Geom& G, const void* canonical,
                        int canonical_is_f64, cudaStream_t st)
{
    if (precision == PREC_F64)
        return recon == 12 ? pack_run<double, 12>(links, G, canonical, canonical_is_f64, st)
                           : pack_run<double, 18>(links, G, canonical, canonical_is_f64, st);
    return recon == 12 ? pack_run<float, 12>(links, G, canonical, canonical_is_f64, st)
                       : pack_run<float, 18>(links, G, canonical, canonical_is_f64, st);
}

cudaError_t launch_unpack(int precision, int recon, const void* links, const Geom& G, void* canonical,
                          int canonical_is_f64, cudaStream_t st)
{
    if (precision == PREC_F64)
        return recon == 12 ? unpack_run<double, 12>(links, G, canonical, canonical_is_f64, st)
                           : unpack_run<double, 18>(links, G, canonical, canonical_is_f64, st);
    return recon == 12 ? unpack_run<float, 12>(links, G, canonical, canonical_is_f64, st)
                       : unpack_run<float, 18>(links, G, canonical, canonical_is_f64, st);
}

template <typename TS, typename TD>
static cudaError_t cast_run(int recon, const void* src, void* dst, const Geom& G, int reproject, int nblocks, cudaStream_t st,
                            const uint32_t* stop)
{
    const uint32_t block = 128;
    const dim3 grid((G.Vh + block - 1) / block, (uint32_t)nblocks, 1);
    if (recon == 12) {
        uniform_carveout(cast_kernel<TS, TD, 12>);
        cast_kernel<TS, TD, 12><<<grid, block, 0, st>>>(static_cast<const TS*>(src), static_cast<TD*>(dst), G, reproject, stop);
    } else {
        uniform_carveout(cast_kernel<TS, TD, 18>);
        cast_kernel<TS, TD, 18><<<grid, block, 0, st>>>(static_cast<const TS*>(src), static_cast<TD*>(dst), G, reproject, stop);
    }
    return cudaGetLastError();
}

cudaError_t launch_cast(int from_precision, int to_precision, int recon, const void* src, void* dst,
                        const Geom& G, int reproject, int nblocks, cudaStream_t st, const uint32_t* stop)
{
    if (from_precision == PREC_F32 && to_precision == PREC_F64) return cast_run<float, double>(recon, src, dst, G, reproject, nblocks, st, stop);
    if (from_precision == PREC_F64 && to_precision == PREC_F32) return cast_run<double, float>(recon, src, dst, G, reproject, nblocks, st, stop);
    if (from_precision == PREC_F64) return cast_run<double, double>(recon, src, dst, G, reproject, nblocks, st, stop);
    return cast_run<float, float>(recon, src, dst, G, reproject, nblocks, st, stop);
}

// ------------------------------------------------------- the accumulated transformation G(x)
// G[parity][chunk][h]: one link-shaped block per parity.  Canonical form: (V,3,3) complex, site-major.
template <typename T, int RECON, typename TC, bool TO_INTERNAL>
__global__ void transform_convert_kernel(T* __restrict__ gtrans, const Geom G, TC* __restrict__ canonical)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 2u * G.Vh) return;
    const uint32_t parity = i >= G.Vh ? 1u : 0u, h = i - parity * G.Vh;
    const Site s = decode_site(G, h, parity);
    TC* c = canonical + (2u * (size_t)h + s.xodd) * 18;
    T* blk = gtrans + (size_t)parity * RECON * padded_vh<T>(G);
    T m[18];
    if (TO_INTERNAL) {
#pragma unroll
        for (int k = 0; k < 18; ++k) m[k] = (T)c[k];
        store_link<RECON>(blk, h, m);
    } else {
        load_link<RECON>(blk, h, m);
        if (RECON == 12) reconstruct_row2(m);
#pragma unroll
        for (int k = 0; k < 18; ++k) c[k] = (TC)m[k];
    }
}

template <typename T, int RECON>
__global__ void transform_identity_kernel(T* __restrict__ gtrans, const Geom G)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 2u * G.Vh) return;
    const uint32_t parity = i >= G.Vh ? 1u : 0u, h = i - parity * G.Vh;
    T m[18];
#pragma unroll
    for (int k = 0; k < 18; ++k) m[k] = T(0);
    m[0] = m[8] = m[16] = T(1);
    store_link<RECON>(gtrans + (size_t)parity * RECON * padded_vh<T>(G), h, m);
}

template <typename T, int RECON, bool TO_INTERNAL>
static cudaError_t transform_convert_run(void* gtrans, const Geom& G, void* canonical, int canonical_is_f64, cudaStream_t st)
{
    const uint32_t n = 2u * G.Vh, block = 128, grid = (n + block - 1) / block;
    if (canonical_is_f64) {
        uniform_carveout(transform_convert_kernel<T, RECON, double, TO_INTERNAL>);
        transform_convert_kernel<T, RECON, double, TO_INTERNAL><<<grid, block, 0, st>>>(static_cast<T*>(gtrans), G, static_cast<double*>(canonical));
    } else {
        uniform_carveout(transform_convert_kernel<T, RECON, float, TO_INTERNAL>);
        transform_convert_kernel<T, RECON, float, TO_INTERNAL><<<grid, block, 0, st>>>(static_cast<T*>(gtrans), G, static_cast<float*>(canonical));
    }
    return cudaGetLastError();
}

template <bool TO_INTERNAL>
static cudaError_t transform_convert(int precision, int recon, void* gtrans, const Geom& G, void* canonical, int is_f64, cudaStream_t st)
{
    if (precision == PREC_F64)
        return recon == 12 ? transform_convert_run<double, 12, TO_INTERNAL>(gtrans, G, canonical, is_f64, st)
                           : transform_convert_run<double, 18, TO_INTERNAL>(gtrans, G, canonical, is_f64, st);
    return recon == 12 ? transform_convert_run<float, 12, TO_INTERNAL>(gtrans, G, canonical, is_f64, st)
                       : transform_convert_run<float, 18, TO_INTERNAL>(gtrans, G, canonical, is_f64, st);
}

cudaError_t launch_transform_pack(int precision, int recon, void* gtrans, const Geom& G, const void* canonical,
                                  int canonical_is_f64, cudaStream_t st)
{
    return transform_convert<true>(precision, recon, gtrans, G, const_cast<void*>(canonical), canonical_is_f64, st);
}

cudaError_t launch_transform_unpack(int precision, int recon, const void* gtrans, const Geom& G, void* canonical,
                                    int canonical_is_f64, cudaStream_t st)
{
    return transform_convert<false>(precision, recon, const_cast<void*>(gtrans), G, canonical, canonical_is_f64, st);
}

cudaError_t launch_transform_identity(int precision, int recon, void* gtrans, const Geom& G, cudaStream_t st)
{
    const uint32_t n = 2u * G.Vh, block = 128, grid = (n + block - 1) / block;
    if (precision == PREC_F64) {
        if (recon == 12) { uniform_carveout(transform_identity_kernel<double, 12>); transform_identity_kernel<double, 12><<<grid, block, 0, st>>>(static_cast<double*>(gtrans), G); }
        else { uniform_carveout(transform_identity_kernel<double, 18>); transform_identity_kernel<double, 18><<<grid, block, 0, st>>>(static_cast<double*>(gtrans), G); }
    } else {
        if (recon == 12) { uniform_carveout(transform_identity_kernel<float, 12>); transform_identity_kernel<float, 12><<<grid, block, 0, st>>>(static_cast<float*>(gtrans), G); }
        else { uniform_carveout(transform_identity_kernel<float, 18>); transform_identity_kernel<float, 18><<<grid, block, 0, st>>>(static_cast<float*>(gtrans), G); }
    }
    return cudaGetLastError();
}

// PAPER.md:43 (eq. 3): dst_mu(x) = G(x) src_mu(x) G(x+mu)^dagger, formed in fp64 whatever the storage
// types.  A transformation accumulated in fp32 has drifted from SU(3) by its rounding; it is
// re-projected (Gram-Schmidt) in fp64 before use, so that the result is gauge equivalent to src to
// fp64 accuracy.  Every link is read and written by the same thread: src may alias dst.
template <typename TG, int RECON>
__device__ __forceinline__ void load_transform_d(const TG* gtrans, const Geom& G, uint32_t parity, uint32_t h, double (&m)[18])
{
    TG u[18];
    load_link<RECON>(gtrans + (size_t)parity * RECON * padded_vh<TG>(G), h, u);
    if (RECON == 12) reconstruct_row2(u);
#pragma unroll
    for (int k = 0; k < 18; ++k) m[k] = (double)u[k];
    if (sizeof(TG) == 4) project_su3(m);
}

template <typename TG, typename TS, typename TD, int RECON>
__global__ void apply_transform_kernel(const TG* __restrict__ gtrans, const TS* src, TD* dst, const Geom G,
                                       const int mu_begin, const int mu_end)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 2u * G.Vh) return;
    const uint32_t parity = i >= G.Vh ? 1u : 0u, h = i - parity * G.Vh;
    const Site s = decode_site(G, h, parity);
    double Gx[18];
    load_transform_d<TG, RECON>(gtrans, G, parity, h, Gx);
    for (int mu = mu_begin; mu < mu_end; ++mu) {
        double U[18], Gf[18], tmp[18], out[18];
        load_full_d<TS, RECON>(src, G, parity, mu, h, U);
        load_transform_d<TG, RECON>(gtrans, G, parity ^ 1u, forward_index(G, s, mu), Gf);
        mul_full(Gx, U, tmp, false);
        mul_full(tmp, Gf, out, true);
        TD o[18];
#pragma unroll
        for (int k = 0; k < 18; ++k) o[k] = (TD)out[k];
        store_link<RECON>(dst + block_offset<TD>(parity, mu, RECON, G), h, o);
    }
}

template <typename TG, typename TS, typename TD>
static cudaError_t apply_run(int recon, const void* gtrans, const void* src, void* dst, const Geom& G, int mu_begin, int mu_end,
                             cudaStream_t st)
{
    const uint32_t n = 2u * G.Vh, block = 128, grid = (n + block - 1) / block;
    if (recon == 12) {
        uniform_carveout(apply_transform_kernel<TG, TS, TD, 12>);
        apply_transform_kernel<TG, TS, TD, 12><<<grid, block, 0, st>>>(static_cast<const TG*>(gtrans), static_cast<const TS*>(src), static_cast<TD*>(dst), G, mu_begin, mu_end);
    } else {
        uniform_carveout(apply_transform_kernel<TG, TS, TD, 18>);
        apply_transform_kernel<TG, TS, TD, 18><<<grid, block, 0, st>>>(static_cast<const TG*>(gtrans), static_cast<const TS*>(src), static_cast<TD*>(dst), G, mu_begin, mu_end);
    }
    return cudaGetLastError();
}

template <typename TG>
static cudaError_t apply_prec(int src_precision, int dst_precision, int recon, const void* gtrans, const void* src, void* dst,
                              const Geom& G, int mu_begin, int mu_end, cudaStream_t st)
{
    if (src_precision == PREC_F64)
        return dst_precision == PREC_F64 ? apply_run<TG, double, double>(recon, gtrans, src, dst, G, mu_begin, mu_end, st)
                                         : apply_run<TG, double, float>(recon, gtrans, src, dst, G, mu_begin, mu_end, st);
    return dst_precision == PREC_F64 ? apply_run<TG, float, double>(recon, gtrans, src, dst, G, mu_begin, mu_end, st)
                                     : apply_run<TG, float, float>(recon, gtrans, src, dst, G, mu_begin, mu_end, st);
}

cudaError_t launch_apply_transform(int g_precision, int src_precision, int dst_precision, int recon,
                                   const void* gtrans, const void* src, void* dst, const Geom& G,
                                   int mu_begin, int mu_end, cudaStream_t st)
{
    return g_precision == PREC_F64 ? apply_prec<double>(src_precision, dst_precision, recon, gtrans, src, dst, G, mu_begin, mu_end, st)
                                   : apply_prec<float>(src_precision, dst_precision, recon, gtrans, src, dst, G, mu_begin, mu_end, st);
}

// ------------------------------------------------------------------------------- Philox KAT
__global__ void philox_kernel(int n, const uint32_t* __restrict__ ctr, const uint32_t* __restrict__ key,
                              uint32_t* __restrict__ out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint32_t w[4];
    philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], key[2 * i], key[2 * i + 1], w);
#pragma unroll
    for (int k = 0; k < 4; ++k) out[4 * i + k] = w[k];
}

cudaError_t launch_philox(int n, const uint32_t* ctr, const uint32_t* key, uint32_t* out, cudaStream_t st)
{
    uniform_carveout(philox_kernel);
    philox_kernel<<<(n + 127) / 128, 128, 0, st>>>(n, ctr, key, out);
    return cudaGetLastError();
}

}  // namespace gf
