// gf_wave.cu -- the streamed sweep: the same site update as gf_sweep.cu, organised for the
// memory system instead of for the register file.
//
// * Persistent blocks.  One PRODUCER warp per block moves the links of a tile -- 32 consecutive sites of one parity:
//   whole x-rows inside one (z,t) plane -- into a ring of shared-memory stages with 1-D TMA bulk copies
//   (cp.async.bulk.shared.global, completion counted by an mbarrier): in the chunked layout block[c][h] every
//   (link, 16-byte chunk) of a tile is ONE contiguous run, forward links and all four backward neighbours alike (the
//   x-neighbour is the same run read with a shifted index, the y-neighbour the run one row down, z and t one plane /
//   one time slice down, periodic wraps are a second run at most).  No tensor map is needed.
// * CONSUMER warps, one thread per site: K(x) is accumulated out of shared memory, the three SU(2) solves run ONCE per
//   site (the register kernel of gf_sweep.cu repeats them in each of the 2-4 lanes that share a site), the links are
//   read from shared memory a second time for g U and U g^dagger and stored to global memory with 128-bit stores.
//   Only K, g and one link are live in registers, so a handful of consumer warps saturates the arithmetic while the
//   ring keeps ~100-200 KB of loads in flight per SM: load latency is decoupled from the arithmetic.
// * Fused iteration (mode 2): ONE launch does both half-sweeps of an iteration in a wavefront over the
//   (t,z) planes -- the parity-1 tiles of plane q are handed out `lag` planes behind the parity-0 tiles -- so that the
//   second touch of every link finds it in the 126 MB L2 and the field crosses the DRAM interface once per iteration
//   instead of twice.  A parity-1 tile needs the parity-0 updates of all its neighbours: its producer waits for the
//   completion counters of the five planes (t,z), (t,z+-1), (t+-1,z), which the consumers of parity-0 tiles publish
//   (release) after their stores.  Tiles are claimed in batches from a global ticket by blocks that are RUNNING, and a
//   block works through its tiles in ticket order, so whatever a block waits for is held by a running block that never
//   waits for a later ticket: no deadlock, whatever the hardware's dispatch order and however many streams share the GPU.
// * Modes 0 / 1: one half-sweep (no dependencies) through the same pipeline.
//
// The links produced are bitwise those of two gf_sweep launches with one lane per site (same arithmetic, same order).
#include "gf_internal.h"

namespace gf {

constexpr uint32_t WAVE_TS = 32;        // sites per tile = one consumer warp
constexpr uint32_t WAVE_BATCH = 4;      // tiles claimed per ticket
constexpr uint32_t WAVE_HEADER = 1024;  // bytes of shared memory in front of the stages (barriers, tile descriptors)

struct TileDesc {
    uint32_t h0;        // first half-index of the tile
    uint32_t plane;     // t * Nz + z
    uint32_t flags;     // bit 0: a tile (0 = the producer is done); bit 1: parity; bit 2: publish completion; bit 3: poisoned
    uint32_t pad;
};

template <typename T, typename TK> struct WaveConsts {
    T* links;
    Geom G;
    uint32_t site_offset;
    int mu0, algo;
    TK omega;
    double p;
    uint32_t key0, key1, counter;
    uint32_t mode;                  // 0 / 1: half-sweep of that parity; 2: fused iteration
    uint32_t M;                     // tiles per plane and parity
    uint32_t planes;                // Nt * Nz
    uint32_t plane_sites;           // sites of one parity in a plane: (Nx/2) * Ny
    uint32_t lag;                   // fused iteration: parity-1 tiles of plane q follow the parity-0 tiles of plane q + lag
    unsigned long long total_tiles;
    unsigned long long* ticket;     // device counter, never reset
    unsigned long long ticket_base;
    uint32_t* done;                 // per plane: parity-0 tiles completed, monotonic over launches
    uint32_t done_target;           // value of done[plane] once all parity-0 tiles of the plane of THIS launch are complete
    uint32_t* error;                // device word: set to 1 if a dependency wait gave up (never expected)
    FastDiv div_M;
};

// ------------------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    while (!mbar_try_wait(bar, parity)) {
    }
}
// global -> shared bulk copy by the TMA unit; `bytes` (a multiple of 16) are counted on `bar` when they have landed
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ uint32_t ld_acquire_gpu(const uint32_t* p)
{
    uint32_t v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release_gpu_add(uint32_t* p, uint32_t v)
{
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t ld_volatile_u32(const uint32_t* p)
{
    uint32_t v;
    asm volatile("ld.volatile.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// ------------------------------------------------------------------------------- the schedule
// Ticket order of the segments (a segment = the M tiles of one plane and parity).  E(q) / O(q): parity-0 / parity-1
// tiles of plane q = t * Nz + z; P planes; D = lag >= Nz + 1; A = D + Nz <= P.
//     E(0) .. E(A-1) | E(k), O(k-D) for k = A .. P-1 | O(P-D) .. O(P-1) | O(0) .. O(Nz-1)
// O(q) with t >= 1 comes after E(q+D), hence after every E it depends on (the latest is E(q+Nz), or a plane of time
// slice 0 when t = Nt-1); the parity-1 tiles of time slice 0 depend on slice Nt-1 and come last.
struct WaveTile {
    uint32_t parity, plane, m;
};

template <typename T, typename TK>
__device__ __forceinline__ WaveTile wave_schedule(const WaveConsts<T, TK>& P, unsigned long long n)
{
    WaveTile w;
    const uint32_t seg = fdiv((uint32_t)n, P.div_M);        // total_tiles < 2^32 (checked on the host)
    w.m = (uint32_t)n - seg * P.M;
    if (P.mode < 2u) {
        w.parity = P.mode;
        w.plane = seg;
        return w;
    }
    const uint32_t D = P.lag, A = D + P.G.nz, B = P.planes - A;
    if (seg < A) {
        w.parity = 0;
        w.plane = seg;
    } else if (seg < A + 2u * B) {
        const uint32_t r = seg - A, k = A + (r >> 1);
        w.parity = r & 1u;
        w.plane = w.parity ? k - D : k;
    } else {
        const uint32_t j = seg - (A + 2u * B);
        w.parity = 1;
        w.plane = j < D ? P.planes - D + j : j - D;
    }
    return w;
}

// ------------------------------------------------------------------------ shared-memory stage
// stage[slot 0..7][chunk][site]: slot mu = U_mu(x), slot 4 + mu = U_mu(x - mu); 16-byte chunks as in global memory
// (fp32 / 18-real: four float4 chunks per link, then the float2 tails of all slots).  Thread i reads chunk c of its
// site at ((slot * CH + c) * 32 + i) * 16: a warp reads 512 contiguous bytes, conflict free.
template <typename T, int RECON> struct StageLayout;
template <int RECON> struct StageLayout<double, RECON> {
    static constexpr int CH16 = RECON / 2, TAIL = 0;
};
template <int RECON> struct StageLayout<float, RECON> {
    static constexpr int CH16 = RECON / 4, TAIL = RECON == 18 ? 1 : 0;
};

template <int RECON>
__device__ __forceinline__ void lds_link(const unsigned char* stage, int slot, uint32_t idx, double (&m)[18])
{
    constexpr int CH = StageLayout<double, RECON>::CH16;
    const double2* p = reinterpret_cast<const double2*>(stage) + (size_t)slot * CH * WAVE_TS + idx;
#pragma unroll
    for (int c = 0; c < CH; ++c) {
        const double2 v = p[c * WAVE_TS];
        m[2 * c] = v.x;
        m[2 * c + 1] = v.y;
    }
}

template <int RECON>
__device__ __forceinline__ void lds_link(const unsigned char* stage, int slot, uint32_t idx, float (&m)[18])
{
    constexpr int CH = StageLayout<float, RECON>::CH16;
    const float4* p = reinterpret_cast<const float4*>(stage) + (size_t)slot * CH * WAVE_TS + idx;
#pragma unroll
    for (int c = 0; c < CH; ++c) {
        const float4 v = p[c * WAVE_TS];
        m[4 * c] = v.x;
        m[4 * c + 1] = v.y;
        m[4 * c + 2] = v.z;
        m[4 * c + 3] = v.w;
    }
    if (RECON == 18) {
        const float2 v = reinterpret_cast<const float2*>(stage + (size_t)8 * CH * WAVE_TS * 16)[slot * WAVE_TS + idx];
        m[16] = v.x;
        m[17] = v.y;
    }
}

// ------------------------------------------------------------------------------ the producer
template <typename T, typename TK, int RECON, int S, int C>
__device__ __forceinline__ void wave_producer(const WaveConsts<T, TK>& P, uint64_t* full, uint64_t* empty, TileDesc* desc,
                                              unsigned char* stages, uint32_t lane)
{
    using L = StageLayout<T, RECON>;
    constexpr uint32_t CHT = L::CH16 + L::TAIL;                                    // runs per link
    constexpr uint32_t STAGE_BYTES = WAVE_TS * 8u * RECON * (uint32_t)sizeof(T);
    const Geom& G = P.G;
    const uint32_t Sh = G.stride[0];                                               // sites of one parity in a time slice
    const unsigned char* base = reinterpret_cast<const unsigned char*>(P.links);
    uint32_t it = 0;
    bool drain = false;                                                            // an error was seen: no more waiting, no more work
    for (;;) {
        unsigned long long b = 0;
        if (lane == 0) b = atomicAdd(P.ticket, (unsigned long long)WAVE_BATCH) - P.ticket_base;
        b = __shfl_sync(0xffffffffu, b, 0);
        if (b >= P.total_tiles) break;
        if (!drain && ld_volatile_u32(P.error) != 0u) drain = true;
        for (unsigned long long n = b; n < b + WAVE_BATCH && n < P.total_tiles; ++n, ++it) {
            const uint32_t slot = it % S, ph = (it / S) & 1u;
            mbar_wait(empty + slot, ph ^ 1u);                                      // the consumers have released the slot
            const WaveTile w = wave_schedule(P, n);
            const uint32_t t = fdiv(w.plane, G.div_nz), z = w.plane - t * G.nz;
            const uint32_t h0 = w.plane * P.plane_sites + w.m * WAVE_TS;
            const uint32_t y0 = fdiv(w.m * WAVE_TS, G.div_nxh);
            if (P.mode == 2u && w.parity == 1u && !drain) {
                // the five planes whose parity-0 updates this tile's links have received
                if (lane < 5u) {
                    uint32_t q = w.plane;
                    if (lane == 1u) q = z + 1u < G.nz ? w.plane + 1u : w.plane + 1u - G.nz;
                    if (lane == 2u) q = z > 0u ? w.plane - 1u : w.plane + G.nz - 1u;
                    if (lane == 3u) q = t + 1u < G.nt ? w.plane + G.nz : z;
                    if (lane == 4u) q = t > 0u ? w.plane - G.nz : w.plane + (G.nt - 1u) * G.nz;
                    for (uint32_t spins = 0; (int32_t)(ld_acquire_gpu(P.done + q) - P.done_target) < 0; ++spins) {
                        __nanosleep(64);
                        if (spins > (1u << 22) || (spins & 1023u) == 1023u && ld_volatile_u32(P.error) != 0u) {
                            *P.error = 1u;                                         // give up: nothing of this tile is stored
                            __threadfence();
                            break;
                        }
                    }
                }
                __syncwarp();
                if (ld_volatile_u32(P.error) != 0u) drain = true;
                // the other blocks' stores (generic proxy) are acquired; the bulk copies below read through the async proxy
                asm volatile("fence.proxy.async;" ::: "memory");
            }
            if (lane == 0) {
                TileDesc d;
                d.h0 = h0;
                d.plane = w.plane;
                d.flags = 1u | (w.parity << 1) | ((P.mode == 2u && w.parity == 0u) ? 4u : 0u) | (drain ? 8u : 0u);
                d.pad = 0;
                desc[slot] = d;
                if (drain) mbar_arrive(full + slot);
                else mbar_expect_tx(full + slot, STAGE_BYTES);
            }
            __syncwarp();
            if (drain) continue;
            unsigned char* stage = stages + (size_t)slot * STAGE_BYTES;
            // runs: (link slot 0..7, chunk); a tile that starts at y = 0 takes its y-neighbours in two runs (slot 8)
            const bool ywrap = y0 == 0u && WAVE_TS > G.nxh;
            const uint32_t nruns = (ywrap ? 9u : 8u) * CHT;
            for (uint32_t id = lane; id < nruns; id += 32u) {
                const uint32_t ls = id / CHT, c = id - ls * CHT;
                uint32_t sl = ls, par = w.parity, hsrc = h0, dst = 0, ns = WAVE_TS;
                if (ls >= 4u) {
                    par ^= 1u;
                    const uint32_t mu = ls & 3u;
                    if (ls == 8u) {                                  // rows 0 .. R-2 of the tile, shifted up by one row
                        sl = 6u;
                        dst = G.nxh;
                        ns = WAVE_TS - G.nxh;
                    } else if (mu == 2u) {
                        if (y0 > 0u) hsrc = h0 - G.nxh;
                        else {
                            hsrc = h0 + G.nxh * (G.ny - 1u);                      // row Ny-1 of the same plane
                            ns = G.nxh < WAVE_TS ? G.nxh : WAVE_TS;
                        }
                    } else if (mu == 3u) {
                        hsrc = z > 0u ? h0 - P.plane_sites : h0 + P.plane_sites * (G.nz - 1u);
                    } else if (mu == 0u) {
                        hsrc = t > 0u ? h0 - Sh : h0 + Sh * (G.nt - 1u);
                    }
                }
                const uint32_t mu = sl & 3u;
                const unsigned char* blk = base + block_offset<T>(par, (int)mu, RECON, G.Vh) * sizeof(T);
                if (c < (uint32_t)L::CH16) {
                    bulk_g2s(stage + ((size_t)(sl * L::CH16 + c) * WAVE_TS + dst) * 16u, blk + ((size_t)c * G.Vh + hsrc) * 16u, ns * 16u,
                             full + slot);
                } else {
                    bulk_g2s(stage + (size_t)8 * L::CH16 * WAVE_TS * 16u + ((size_t)sl * WAVE_TS + dst) * 8u,
                             blk + (size_t)16 * G.Vh * sizeof(T) + (size_t)hsrc * 8u, ns * 8u, full + slot);
                }
            }
        }
    }
    // one empty descriptor per consumer warp: consumer w takes the ring entries it = w (mod C)
    for (int k = 0; k < C; ++k, ++it) {
        const uint32_t slot = it % S, ph = (it / S) & 1u;
        mbar_wait(empty + slot, ph ^ 1u);
        if (lane == 0) {
            desc[slot].flags = 0;
            mbar_arrive(full + slot);
        }
        __syncwarp();
    }
}

// ------------------------------------------------------------------------------ the consumers
template <typename T, typename TK, int RECON, int S, int C>
__device__ __forceinline__ void wave_consumer(const WaveConsts<T, TK>& P, uint64_t* full, uint64_t* empty, const TileDesc* desc,
                                              const unsigned char* stages, uint32_t warp, uint32_t lane)
{
    constexpr uint32_t STAGE_BYTES = WAVE_TS * 8u * RECON * (uint32_t)sizeof(T);
    constexpr int ROWS = RECON == 12 ? 2 : 3;
    constexpr uint32_t NONE = 0xffffffffu;
    const Geom& G = P.G;
    uint32_t pending = NONE;                    // plane of a finished parity-0 tile whose completion is not published yet
    for (uint32_t it = warp;; it += C) {
        const uint32_t slot = it % S, ph = (it / S) & 1u;
        if (!mbar_try_wait(full + slot, ph)) {
            // nothing to do yet: publish now (a producer, possibly this block's, may be waiting for exactly this count)
            if (pending != NONE) {
                __syncwarp();
                if (lane == 0) red_release_gpu_add(P.done + pending, 1u);
                pending = NONE;
            }
            mbar_wait(full + slot, ph);
        }
        const TileDesc d = desc[slot];
        if (!(d.flags & 1u)) break;
        if (d.flags & 8u) {                     // poisoned (an error elsewhere): nothing is computed or stored
            __syncwarp();
            if (lane == 0) mbar_arrive(empty + slot);
            continue;
        }
        const uint32_t parity = (d.flags >> 1) & 1u;
        const uint32_t h = d.h0 + lane;
        const unsigned char* stage = stages + (size_t)slot * STAGE_BYTES;
        const Site s = decode_site(G, h, parity);
        uint32_t hb[4];
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) hb[mu] = backward_index(G, s, mu);
        const uint32_t ixb = hb[1] - d.h0;      // the x-neighbour sits in the same row, hence in the same run

        // a3: K(x) = sum_mu [U_mu(x) + U_mu(x-mu)^dagger]  (eq. 8)
        TK K[18];
#pragma unroll
        for (int k = 0; k < 18; ++k) K[k] = TK(0);
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            if (mu >= P.mu0) {
                T Uf[18], Ub[18];
                lds_link<RECON>(stage, mu, lane, Uf);
                lds_link<RECON>(stage, 4 + mu, mu == 1 ? ixb : lane, Ub);
                if (RECON == 12) {
                    reconstruct_row2(Uf);
                    reconstruct_row2(Ub);
                }
#pragma unroll
                for (int a = 0; a < 3; ++a)
#pragma unroll
                    for (int b = 0; b < 3; ++b) {
                        GF_RE(K, a, b) += (TK)GF_RE(Uf, a, b) + (TK)GF_RE(Ub, b, a);
                        GF_IM(K, a, b) += (TK)GF_IM(Uf, a, b) - (TK)GF_IM(Ub, b, a);
                    }
            }
        }

        // a5: the stochastic-relaxation draws
        bool sq0 = false, sq1 = false, sq2 = false;
        if (P.algo == ALGO_STOCHASTIC) {
            uint32_t w[4];
            philox4x32_10(P.site_offset + 2u * h + s.xodd, 0u, P.mode == 2u ? P.counter + parity : P.counter, 0u, P.key0, P.key1, w);
            sq0 = (double)(w[0] >> 8) * (1.0 / 16777216.0) < P.p;
            sq1 = (double)(w[1] >> 8) * (1.0 / 16777216.0) < P.p;
            sq2 = (double)(w[2] >> 8) * (1.0 / 16777216.0) < P.p;
        }

        // a4: the three SU(2) subgroups, once per site
        TK gk[18];
        solve_site(K, P.algo, P.omega, sq0, sq1, sq2, gk);
        T g[18];
#pragma unroll
        for (int k = 0; k < 18; ++k) g[k] = (T)gk[k];

        // the previous tile's stores left long ago: publishing them now costs no waiting
        if (pending != NONE) {
            __syncwarp();
            if (lane == 0) red_release_gpu_add(P.done + pending, 1u);
            pending = NONE;
        }

        // a6: U_mu(x) <- g U_mu(x),  U_mu(x-mu) <- U_mu(x-mu) g^dagger  (eq. 3)
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            T U[18], out[18];
            lds_link<RECON>(stage, mu, lane, U);
            if (RECON == 12) reconstruct_row2(U);
            mul_g_U<ROWS>(g, U, out);
            store_link<RECON>(P.links + block_offset<T>(parity, mu, RECON, G.Vh), G.Vh, h, out);
            lds_link<RECON>(stage, 4 + mu, mu == 1 ? ixb : lane, U);
            mul_U_gdag<ROWS>(U, g, out);
            store_link<RECON>(P.links + block_offset<T>(parity ^ 1u, mu, RECON, G.Vh), G.Vh, hb[mu], out);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(empty + slot);                   // the stage may be refilled
        if (d.flags & 4u) pending = d.plane;
    }
    if (pending != NONE) {
        __syncwarp();
        if (lane == 0) red_release_gpu_add(P.done + pending, 1u);
    }
}

template <typename T, typename TK, int RECON, int S, int C>
__global__ void __launch_bounds__(32 * (C + 1), 1) wave_kernel(const WaveConsts<T, TK> P)
{
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem);
    uint64_t* empty = full + S;
    TileDesc* desc = reinterpret_cast<TileDesc*>(empty + S);
    static_assert(S * (8 + 8 + sizeof(TileDesc)) <= WAVE_HEADER, "header too small");
    unsigned char* stages = smem + WAVE_HEADER;
    if (threadIdx.x == 0) {
        for (int s = 0; s < S; ++s) {
            mbar_init(full + s, 1);
            mbar_init(empty + s, 1);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31u;
    if (warp == (uint32_t)C) wave_producer<T, TK, RECON, S, C>(P, full, empty, desc, stages, lane);
    else wave_consumer<T, TK, RECON, S, C>(P, full, empty, desc, stages, warp, lane);
}

// --------------------------------------------------------------------------------- launching
// stages x consumer warps per storage variant: the ring fills the shared memory of an SM (227 KB per block)
#ifndef GF_WAVE_CFG
#define GF_WAVE_CFG_F64_18 6, 4
#define GF_WAVE_CFG_F64_12 8, 5
#define GF_WAVE_CFG_F32_18 10, 6
#define GF_WAVE_CFG_F32_12 12, 6
#endif
template <typename T, int RECON> struct WaveCfg;
template <> struct WaveCfg<double, 18> { static constexpr int cfg[2] = {GF_WAVE_CFG_F64_18}; };
template <> struct WaveCfg<double, 12> { static constexpr int cfg[2] = {GF_WAVE_CFG_F64_12}; };
template <> struct WaveCfg<float, 18> { static constexpr int cfg[2] = {GF_WAVE_CFG_F32_18}; };
template <> struct WaveCfg<float, 12> { static constexpr int cfg[2] = {GF_WAVE_CFG_F32_12}; };

bool wave_supported(const Geom& G)
{
    // a tile = 32 sites = whole x-rows inside one plane; runs of the fp32 tail array must stay 16-byte aligned
    const uint32_t plane = G.nxh * G.ny;
    return G.nxh >= 2 && G.nxh % 2u == 0 && WAVE_TS % G.nxh == 0 && plane % WAVE_TS == 0;
}

uint32_t wave_stages(int precision, int recon)
{
    if (precision == PREC_F64) return recon == 12 ? WaveCfg<double, 12>::cfg[0] : WaveCfg<double, 18>::cfg[0];
    return recon == 12 ? WaveCfg<float, 12>::cfg[0] : WaveCfg<float, 18>::cfg[0];
}

uint32_t wave_tiles_per_plane(const Geom& G) { return G.nxh * G.ny / WAVE_TS; }

uint32_t wave_ticket_advance(const WaveArgs& a)
{
    // every block fails exactly one claim; the successful claims cover the tiles in batches
    const unsigned long long total = wave_total_tiles(a);
    return (uint32_t)(((total + WAVE_BATCH - 1) / WAVE_BATCH + (unsigned long long)a.num_ctas) * WAVE_BATCH);
}

unsigned long long wave_total_tiles(const WaveArgs& a)
{
    const unsigned long long per_parity = (unsigned long long)a.G.Vh / WAVE_TS;
    return a.mode == 2 ? 2ull * per_parity : per_parity;
}

template <typename T, typename TK, int RECON>
static cudaError_t launch_wave_t(const WaveArgs& a, cudaStream_t st)
{
    constexpr int S = WaveCfg<T, RECON>::cfg[0], C = WaveCfg<T, RECON>::cfg[1];
    constexpr size_t smem = WAVE_HEADER + (size_t)S * WAVE_TS * 8u * RECON * sizeof(T);
    static_assert(smem <= 232448, "the ring does not fit the shared memory of an SM");
    WaveConsts<T, TK> P;
    P.links = static_cast<T*>(a.links);
    P.G = a.G;
    P.site_offset = a.site_offset;
    P.mu0 = a.mu0;
    P.algo = a.algo;
    P.omega = (TK)a.omega;
    P.p = a.p;
    P.key0 = a.key0;
    P.key1 = a.key1;
    P.counter = a.counter;
    P.mode = (uint32_t)a.mode;
    P.plane_sites = a.G.nxh * a.G.ny;
    P.M = P.plane_sites / WAVE_TS;
    P.planes = a.G.nt * a.G.nz;
    P.lag = a.lag;
    P.total_tiles = wave_total_tiles(a);
    P.ticket = a.ticket;
    P.ticket_base = a.ticket_base;
    P.done = a.done;
    P.done_target = a.done_target;
    P.error = a.error;
    P.div_M = make_fastdiv(P.M);
    auto kernel = wave_kernel<T, TK, RECON, S, C>;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kernel<<<a.num_ctas, 32 * (C + 1), smem, st>>>(P);
    return cudaGetLastError();
}

cudaError_t launch_wave(int precision, int solver_f64, int recon, const WaveArgs& a, cudaStream_t st)
{
    if (!wave_supported(a.G) || a.num_ctas < 1) return cudaErrorInvalidValue;
    if (precision == PREC_F64)
        return recon == 12 ? launch_wave_t<double, double, 12>(a, st) : launch_wave_t<double, double, 18>(a, st);
    if (solver_f64) return recon == 12 ? launch_wave_t<float, double, 12>(a, st) : launch_wave_t<float, double, 18>(a, st);
    return recon == 12 ? launch_wave_t<float, float, 12>(a, st) : launch_wave_t<float, float, 18>(a, st);
}

}  // namespace gf
