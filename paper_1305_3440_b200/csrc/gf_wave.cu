// gf_wave.cu -- the streamed sweep: the same site update as gf_sweep.cu, organised for the
// memory system instead of for the register file.
//
// * Persistent blocks.  One PRODUCER warp per block moves the links of a tile -- the TW = 32 (fp64) or 64 (fp32)
//   consecutive sites of one layout tile: whole x-rows inside one (z,t) plane -- into a ring of shared-memory stages
//   with 1-D TMA bulk copies (cp.async.bulk.shared.global, completion counted by an mbarrier).  In the tiled layout
//   (gf_device.cuh) all chunks of one link for one tile are ONE contiguous run of 4608 / 3072 bytes, so a stage is
//   nine requests: the four forward links, and for the backward neighbours the tile itself (x: same run read with a
//   shifted index; y: rows 1.. of the tile), the tile holding the row below (y), the tile one plane down (z) and one
//   time slice down (t), periodic wraps included.  No tensor map is needed.  (Per-chunk runs of 512 bytes were
//   measured first: a bulk copy costs ~35 ns of TMA time whatever its size, profiles/r2_tma_request_size.txt.)
// * CONSUMER warps (two per stage) run the site update of the register kernel -- one lane per site in fp32, two in
//   fp64 -- but take their links from shared memory instead of global memory and hand the stage back as soon as the
//   links are in registers: the ring only covers the latency of the loads, ~200 KB in flight per SM whatever the
//   arithmetic does, and a consumer never waits for DRAM.  Results go to global memory with 128-bit stores.
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
// The links produced are bitwise those of two gf_sweep launches with one (fp32) / two (fp64) lanes per site.
#include "gf_internal.h"

namespace gf {

constexpr uint32_t WAVE_SLOTS = 9;      // link tiles per stage
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
    uint32_t tiles_per_block;       // layout tiles in one field[parity][mu] block
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
// A stage holds WAVE_SLOTS link tiles exactly as they lie in global memory ([chunk][site] inside the tile), so the
// consumers read them with the same load_link as the register kernel (thread i reads chunk c at (c * TW + i) * 16:
// a warp reads 512 contiguous bytes, conflict free).  Slots: mu = U_mu(x); 4 + mu = U_mu(x - mu) with 4 = the tile one
// time slice down, 5 = this tile (x-neighbours), 6 = this tile (y-neighbours of rows 1..), 7 = one plane down,
// 8 = the tile holding the row below this tile's first row.
template <typename T, int RECON> struct StageLayout {
    static constexpr uint32_t LINK_BYTES = TileUnits<T, RECON>::value * 16u;          // one link tile: 4608 or 3072 bytes
    static constexpr uint32_t STAGE_BYTES = WAVE_SLOTS * LINK_BYTES;
};

template <typename T, int RECON>
__device__ __forceinline__ const T* stage_slot(const unsigned char* stage, uint32_t slot)
{
    return reinterpret_cast<const T*>(stage + (size_t)slot * StageLayout<T, RECON>::LINK_BYTES);
}

// ------------------------------------------------------------------------------ the producer
template <typename T, typename TK, int RECON, int S, int C>
__device__ __forceinline__ void wave_producer(const WaveConsts<T, TK>& P, uint64_t* full, uint64_t* empty, TileDesc* desc,
                                              unsigned char* stages, uint32_t lane)
{
    using L = StageLayout<T, RECON>;
    constexpr uint32_t TW = Tile<T>::W;
    const Geom& G = P.G;
    const unsigned char* base = reinterpret_cast<const unsigned char*>(P.links);
    const uint32_t tiles_slice = P.M * G.nz;                                        // tiles of one parity in a time slice
    uint32_t it = 0;
    uint32_t verified = 0xffffffffu;                                               // plane whose dependencies this block has seen complete
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
            const uint32_t tile = w.plane * P.M + w.m;                             // layout tile inside a field block
            const bool first_rows = w.m == 0u;                                     // the tile starts at y = 0
            if (P.mode == 2u && w.parity == 1u && !drain && w.plane != verified) {
                // the five planes whose parity-0 updates this tile's links have received
                if (lane < 5u) {
                    uint32_t q = w.plane;
                    if (lane == 1u) q = z + 1u < G.nz ? w.plane + 1u : w.plane + 1u - G.nz;
                    if (lane == 2u) q = z > 0u ? w.plane - 1u : w.plane + G.nz - 1u;
                    if (lane == 3u) q = t + 1u < G.nt ? w.plane + G.nz : z;
                    if (lane == 4u) q = t > 0u ? w.plane - G.nz : w.plane + (G.nt - 1u) * G.nz;
                    for (uint32_t spins = 0; (int32_t)(ld_acquire_gpu(P.done + q) - P.done_target) < 0; ++spins) {
                        __nanosleep(64);
                        if (spins > (1u << 22) || ((spins & 1023u) == 1023u && ld_volatile_u32(P.error) != 0u)) {
                            *P.error = 1u;                                         // give up: nothing of this tile is stored
                            __threadfence();
                            break;
                        }
                    }
                }
                __syncwarp();
                if (ld_volatile_u32(P.error) != 0u) drain = true;
                verified = w.plane;                                                // the tiles of a plane share their five counters
                // the other blocks' stores (generic proxy) are acquired; the bulk copies below read through the async proxy
                asm volatile("fence.proxy.async;" ::: "memory");
            }
            const bool own_y = G.nxh < TW;                                         // rows 1.. of the tile have their y-neighbours in it
            if (lane == 0) {
                TileDesc d;
                d.h0 = tile * TW;
                d.plane = w.plane;
                d.flags = 1u | (w.parity << 1) | ((P.mode == 2u && w.parity == 0u) ? 4u : 0u) | (drain ? 8u : 0u);
                d.pad = 0;
                desc[slot] = d;
                if (drain) mbar_arrive(full + slot);
                else mbar_expect_tx(full + slot, (own_y ? 9u : 8u) * L::LINK_BYTES);
            }
            __syncwarp();
            if (drain || lane >= WAVE_SLOTS || (lane == 6u && !own_y)) continue;
            // lane = slot: one request per link tile
            uint32_t par = w.parity, mu = lane & 3u, src = tile;
            if (lane >= 4u) {
                par ^= 1u;
                if (lane == 4u) src = t > 0u ? tile - tiles_slice : tile + tiles_slice * (G.nt - 1u);
                else if (lane == 7u) src = z > 0u ? tile - P.M : tile + P.M * (G.nz - 1u);
                else if (lane == 8u) {
                    mu = 2u;
                    src = first_rows ? tile + P.M - 1u : tile - 1u;               // the tile whose last row lies below ours
                }
            }
#ifdef GF_WAVE_DEBUG_NOTMA
            // bottleneck probe: the consumers alone (they compute on whatever the stage holds)
            asm volatile("mbarrier.complete_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(full + slot)), "r"(L::LINK_BYTES) : "memory");
#else
            bulk_g2s(stages + (size_t)slot * L::STAGE_BYTES + (size_t)lane * L::LINK_BYTES,
                     base + block_offset<T>(par, (int)mu, RECON, G) * sizeof(T) + (size_t)src * L::LINK_BYTES, L::LINK_BYTES, full + slot);
#endif
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
// Lanes per site and warps per tile.  fp64: two lanes per site (each holds two directions, as in the register kernel),
// 16 sites per warp, two warps per 32-site tile.  fp32: one lane per site, two warps per 64-site tile.
template <typename T> struct WaveShape {
    static constexpr int L = sizeof(T) == 8 ? 2 : 1;
    static constexpr uint32_t SPW = 32u / L;                    // sites per warp
    static constexpr uint32_t CW = Tile<T>::W / SPW;            // consumer warps per stage
};

template <typename T, typename TK, int RECON, int S, int C>
__device__ __forceinline__ void wave_consumer(const WaveConsts<T, TK>& P, uint64_t* full, uint64_t* empty, const TileDesc* desc,
                                              const unsigned char* stages, uint32_t warp, uint32_t lane)
{
    using SL = StageLayout<T, RECON>;
    constexpr uint32_t TW = Tile<T>::W;
    constexpr int L = WaveShape<T>::L, ND = 4 / L;
    constexpr uint32_t SPW = WaveShape<T>::SPW, CW = WaveShape<T>::CW;
    constexpr int ROWS = RECON == 12 ? 2 : 3;
    constexpr uint32_t NONE = 0xffffffffu;
    const Geom& G = P.G;
    const uint32_t group = warp / CW, sub = warp % CW;
    const uint32_t i = sub * SPW + lane % SPW;  // site of this lane inside a tile
    const int j = lane / SPW;                   // which directions it holds: mu = j * ND ..
    uint32_t pending = NONE;                    // plane of a finished parity-0 tile whose completion is not published yet
    for (uint32_t it = group;; it += C) {
        const uint32_t slot = it % S, ph = (it / S) & 1u;
        // A parity wait may run at most one phase ahead of its barrier.  The previous fill of this slot may have been
        // consumed by ANOTHER group (C does not divide S), and bulk copies complete out of order under load, so this
        // warp first makes sure that fill was released -- which implies it landed -- before it waits for its own.
        const bool ready = (it < (uint32_t)S || mbar_try_wait(empty + slot, ph ^ 1u)) && mbar_try_wait(full + slot, ph);
        if (!ready) {
            // nothing to do yet: publish now (a producer, possibly this block's, may be waiting for exactly this count)
            if (pending != NONE) {
                __syncwarp();
                if (lane == 0) red_release_gpu_add(P.done + pending, 1u);
                pending = NONE;
            }
            if (it >= (uint32_t)S) mbar_wait(empty + slot, ph ^ 1u);
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
        const unsigned char* stage = stages + (size_t)slot * SL::STAGE_BYTES;
        const uint32_t h = d.h0 + i;
        const Site s = decode_site(G, h, parity);

        // a2: this lane's links out of the stage into registers, then the stage goes back to the producer: the ring
        // only has to cover the latency of the loads, not the arithmetic
        T Uf[ND][18], Ub[ND][18];
        uint32_t hb[ND];
#pragma unroll
        for (int dd = 0; dd < ND; ++dd) {
            const int mu = j * ND + dd;
            hb[dd] = backward_index(G, s, mu);
            load_link<RECON>(stage_slot<T, RECON>(stage, mu), i, Uf[dd]);
            // where the backward neighbour sits in the stage: x in the same row of this tile, y one row down
            uint32_t bslot = 4u + (uint32_t)mu, bi = i;
            if (mu == 1) bi = hb[dd] - d.h0;
            if (mu == 2) {
                bslot = i >= G.nxh ? 6u : 8u;
                bi = i >= G.nxh ? i - G.nxh : TW - G.nxh + i;
            }
            load_link<RECON>(stage_slot<T, RECON>(stage, bslot), bi, Ub[dd]);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(empty + slot);       // release: the loads above are performed before it
#ifdef GF_WAVE_DEBUG_NOCOMPUTE
        if (Uf[0][0] != T(12345.678)) continue;          // bottleneck probe: the producer / TMA path alone
#endif

        // a3: K(x) = sum_mu [U_mu(x) + U_mu(x-mu)^dagger]  (eq. 8); 12-real: the third rows are formed
        // for K and dropped (as in the register kernel's lazy variant)
        TK K[18];
#pragma unroll
        for (int k = 0; k < 18; ++k) K[k] = TK(0);
#pragma unroll
        for (int dd = 0; dd < ND; ++dd) {
            const int mu = j * ND + dd;
            if (mu >= P.mu0) {
                T rf[6], rb[6];
                if (RECON == 12) {
                    row2_of(Uf[dd], rf);
                    row2_of(Ub[dd], rb);
                }
#pragma unroll
                for (int a = 0; a < 3; ++a)
#pragma unroll
                    for (int b = 0; b < 3; ++b) {
                        const T fr = (RECON == 18 || a < 2) ? GF_RE(Uf[dd], a, b) : rf[2 * b];
                        const T fi = (RECON == 18 || a < 2) ? GF_IM(Uf[dd], a, b) : rf[2 * b + 1];
                        const T br = (RECON == 18 || b < 2) ? GF_RE(Ub[dd], b, a) : rb[2 * a];
                        const T bi = (RECON == 18 || b < 2) ? GF_IM(Ub[dd], b, a) : rb[2 * a + 1];
                        GF_RE(K, a, b) += (TK)fr + (TK)br;
                        GF_IM(K, a, b) += (TK)fi - (TK)bi;
                    }
            }
        }
#pragma unroll
        for (uint32_t off = SPW; off < 32u; off <<= 1) {
#pragma unroll
            for (int k = 0; k < 18; ++k) K[k] += __shfl_xor_sync(0xffffffffu, K[k], off);
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

        // a4: the three SU(2) subgroups
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
        for (int dd = 0; dd < ND; ++dd) {
            const int mu = j * ND + dd;
            T out[18];
            if (RECON == 12) {
                forget(GF_RE(Uf[dd], 0, 1));
                forget(GF_RE(Uf[dd], 0, 2));
                reconstruct_row2(Uf[dd]);
            }
            mul_g_U<ROWS>(g, Uf[dd], out);
            store_link<RECON>(P.links + block_offset<T>(parity, mu, RECON, G), h, out);
            mul_U_gdag<ROWS>(Ub[dd], g, out);
            store_link<RECON>(P.links + block_offset<T>(parity ^ 1u, mu, RECON, G), hb[dd], out);
        }
        if (d.flags & 4u) pending = d.plane;
    }
    if (pending != NONE) {
        __syncwarp();
        if (lane == 0) red_release_gpu_add(P.done + pending, 1u);
    }
}

template <typename T, typename TK, int RECON, int S, int C>
__global__ void __launch_bounds__(32 * (C * (int)WaveShape<T>::CW + 1), 1) wave_kernel(const WaveConsts<T, TK> P)
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
            mbar_init(empty + s, WaveShape<T>::CW);                 // every consumer warp of the stage releases it
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31u;
    constexpr uint32_t CW = WaveShape<T>::CW;
    if (warp == (uint32_t)C * CW) wave_producer<T, TK, RECON, S, C>(P, full, empty, desc, stages, lane);
    else wave_consumer<T, TK, RECON, S, C>(P, full, empty, desc, stages, warp, lane);
}

// --------------------------------------------------------------------------------- launching
// stages x consumer warps per storage variant: the ring fills the shared memory of an SM (227 KB per block)
#ifndef GF_WAVE_S18
#define GF_WAVE_S18 5
#endif
#ifndef GF_WAVE_S12
#define GF_WAVE_S12 8
#endif
#ifndef GF_WAVE_C
#define GF_WAVE_C 3      // registers are allocated per four warps: 3 groups x 2 warps + the producer = 7 warps leave 255 registers per thread
#endif
#define GF_WAVE_CFG_F64_18 GF_WAVE_S18, GF_WAVE_C
#define GF_WAVE_CFG_F64_12 GF_WAVE_S12, GF_WAVE_C
#define GF_WAVE_CFG_F32_18 GF_WAVE_S18, GF_WAVE_C
#define GF_WAVE_CFG_F32_12 GF_WAVE_S12, GF_WAVE_C
template <typename T, int RECON> struct WaveCfg;
template <> struct WaveCfg<double, 18> { static constexpr int cfg[2] = {GF_WAVE_CFG_F64_18}; };
template <> struct WaveCfg<double, 12> { static constexpr int cfg[2] = {GF_WAVE_CFG_F64_12}; };
template <> struct WaveCfg<float, 18> { static constexpr int cfg[2] = {GF_WAVE_CFG_F32_18}; };
template <> struct WaveCfg<float, 12> { static constexpr int cfg[2] = {GF_WAVE_CFG_F32_12}; };

bool wave_supported(const Geom& G, int precision)
{
    // a layout tile (32 sites in fp64, 64 in fp32) must be whole x-rows inside one (z,t) plane
    const uint32_t plane = G.nxh * G.ny, TW = precision == PREC_F64 ? Tile<double>::W : Tile<float>::W;
    return TW % G.nxh == 0 && plane % TW == 0;
}

uint32_t wave_stages(int precision, int recon)
{
    if (precision == PREC_F64) return recon == 12 ? WaveCfg<double, 12>::cfg[0] : WaveCfg<double, 18>::cfg[0];
    return recon == 12 ? WaveCfg<float, 12>::cfg[0] : WaveCfg<float, 18>::cfg[0];
}

uint32_t wave_tiles_per_plane(const Geom& G, int precision)
{
    return G.nxh * G.ny / (precision == PREC_F64 ? Tile<double>::W : Tile<float>::W);
}

// what a fused launch adds to every done[plane]: one count per consumer warp (two per tile) of its parity-0 tiles
uint32_t wave_counts_per_plane(const Geom& G, int precision) { return 2u * wave_tiles_per_plane(G, precision); }



uint32_t wave_ticket_advance(const WaveArgs& a)
{
    // every block fails exactly one claim; the successful claims cover the tiles in batches
    const unsigned long long total = wave_total_tiles(a);
    return (uint32_t)(((total + WAVE_BATCH - 1) / WAVE_BATCH + (unsigned long long)a.num_ctas) * WAVE_BATCH);
}

unsigned long long wave_total_tiles(const WaveArgs& a)
{
    const unsigned long long per_parity = (unsigned long long)a.G.Vh / (a.precision == PREC_F64 ? Tile<double>::W : Tile<float>::W);
    return a.mode == 2 ? 2ull * per_parity : per_parity;
}

template <typename T, typename TK, int RECON>
static cudaError_t launch_wave_t(const WaveArgs& a, cudaStream_t st)
{
    constexpr int S = WaveCfg<T, RECON>::cfg[0], C = WaveCfg<T, RECON>::cfg[1];
    constexpr size_t smem = WAVE_HEADER + (size_t)S * StageLayout<T, RECON>::STAGE_BYTES;
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
    P.M = P.plane_sites / Tile<T>::W;
    P.tiles_per_block = a.G.Vh / Tile<T>::W;
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
    kernel<<<a.num_ctas, 32 * (C * (int)WaveShape<T>::CW + 1), smem, st>>>(P);
    return cudaGetLastError();
}

cudaError_t launch_wave(int precision, int solver_f64, int recon, const WaveArgs& a, cudaStream_t st)
{
    if (!wave_supported(a.G, precision) || a.num_ctas < 1) return cudaErrorInvalidValue;
    if (precision == PREC_F64)
        return recon == 12 ? launch_wave_t<double, double, 12>(a, st) : launch_wave_t<double, double, 18>(a, st);
    if (solver_f64) return recon == 12 ? launch_wave_t<float, double, 12>(a, st) : launch_wave_t<float, double, 18>(a, st);
    return recon == 12 ? launch_wave_t<float, float, 12>(a, st) : launch_wave_t<float, float, 18>(a, st);
}

}  // namespace gf
