// gf_sweep.cu -- the checkerboard relaxation half-sweep, the hot kernel.
//
// Traffic: a half-sweep reads and writes every link exactly once (the V/2 active sites each own
// 4 forward links and touch the 4 backward links U_mu(x-mu), which are stored on the other
// parity), so the algorithmic bytes per site-update are 16 * RECON * sizeof(T) and the kernel is
// HBM bound (0.9-2.8 flop/byte).  No tensor cores: there is no dense contraction here.
//
// Mapping: L = 1, 2 or 4 lanes cooperate on one site.  Lane j of a site owns the directions
// mu = j*(4/L) .. and keeps U_mu(x) and U_mu(x-mu) in registers (fp64 with L = 1 would need 288
// registers for the links alone).  A warp covers S = 32/L consecutive half-indices; lanes with
// the same j are contiguous in h, so every 128-bit load instruction of a warp touches L fully
// used contiguous runs of S*16 bytes.  The partial K's are combined with an xor-butterfly of
// warp shuffles (bitwise identical in all lanes, additions commute), every lane then computes
// the same g(x) redundantly and applies it to its own links.  The paper's kernel used 8 threads
// per site through shared memory; that is prior art, not this design.
#include "gf_internal.h"

namespace gf {

template <typename T, typename TK> struct SweepConsts {
    T* links;
    T* gtrans;              // MODE > 0: the accumulated transformation G[parity][chunk][h], else unused
    const uint16_t* slice_list;    // Coulomb slice freezing: the launch covers only the listed time slices; NULL = all
    uint32_t n_sites;              // sites of the active parity the launch covers: Vh, or entries of slice_list x G.sh
    T* prev_links;          // slab decomposition in t: field holding U_0(x-0) of the sites with local t = 0 (the rank
                            // below; this rank's own field when there is one slab, which is the periodic wrap)
    uint32_t site_offset;   // global index of this slab's first site (Philox counter word 0)
    Geom G;
    uint32_t parity;
    int mu0, algo;
    TK omega;
    double p;
    uint32_t key0, key1, counter;
    uint32_t reverse;       // 1: blocks walk the lattice from the last site to the first
    const uint32_t* stop;   // see SweepArgs
};

template <typename T>
__device__ __forceinline__ T shfl_xor_T(T v, int mask)
{
    return __shfl_xor_sync(0xffffffffu, v, mask);
}

// T: storage type and the type of the 3x3 products of step a6; TK: type in which K(x) is
// accumulated and the SU(2) solves run (TK = double with T = float costs no bandwidth and removes
// the amplification of fp32 rounding at sites with a small |v|).
// MODE_ACC: also record the transformation, G(x) <- g(x) G(x) (one more matrix read and written per
// site-update, +12.5 % traffic); done by the lane that owns mu = 0.
// MODE_DEFER (Coulomb gauge only, where the temporal links enter neither K nor F nor theta): record
// G(x) and leave U_0(x), U_0(x-0) alone -- 6 links + G instead of 8 links per site-update, -12.5 %
// traffic; U_0(x) <- G(x) U_0(x) G(x+0)^dagger is applied once at the end (gf_coulomb_finish).
enum { MODE_PLAIN = 0, MODE_ACC = 1, MODE_DEFER = 2 };

// 1: half-sweeps are launched with programmatic stream serialisation (see sweep_body); 0: plain stream order
#ifndef GF_PDL
#define GF_PDL 1
#endif

// 0: the half-sweeps ignore the stop word of the run-ahead fix loop (for A/B timing of the sweeps only: gf_fix_until
// then needs gf_set_fix_runahead(ctx, 0))
#ifndef GF_STOP_CHECK
#define GF_STOP_CHECK 1
#endif

// bit L set: the L-lanes-per-site kernel of that storage type is "lazy".  Measured at 32^4 (sustained runs under the
// power cap, profiles/r2_tune_f64_12.txt): fp64 with one or two lanes per site goes from 226 to 166 registers (L = 2) and
// from 81 % to 100 % of the HBM peak; with four lanes it changes nothing.
#ifndef GF_LAZY12_F64
#define GF_LAZY12_F64 6
#endif
#ifndef GF_LAZY12_F32
#define GF_LAZY12_F32 0
#endif
// which 12-real variants drop the third rows between K(x) and the update (see sweep_body)
template <typename T, int L> struct Lazy12 {
    static constexpr bool value = sizeof(T) == 8 ? (GF_LAZY12_F64 >> L) & 1 : (GF_LAZY12_F32 >> L) & 1;
};

template <typename T, typename TK, int RECON, int L, int MODE>
__device__ __forceinline__ void sweep_body(const SweepConsts<T, TK>& P)
{
    constexpr int S = 32 / L;    // sites per warp
    constexpr int ND = 4 / L;    // directions per lane
    constexpr int ROWS = RECON == 12 ? 2 : 3;
    const Geom& G = P.G;
    const uint32_t lane = threadIdx.x & 31u;
    // Alternate half-sweeps walk the lattice in opposite directions (blocks are dispatched in
    // ascending blockIdx order): the launch starts on the sites the previous one finished with,
    // whose links are still in the 126 MB L2.  The result does not depend on the order.
#if GF_PDL
    // Programmatic dependent launch: the next half-sweep of the stream may be scheduled onto SMs as the blocks of this
    // one drain; its blocks wait below, before their first access to global memory, until this grid has completed and
    // its stores are visible.  What overlaps is launch latency and block start-up, never two half-sweeps' accesses.
    asm volatile("griddepcontrol.launch_dependents;");
#endif
    const uint32_t bid = P.reverse ? gridDim.x - 1u - blockIdx.x : blockIdx.x;
    const uint32_t parity = P.parity, counter = P.counter;
    const uint32_t warp = (bid * blockDim.x + threadIdx.x) >> 5;
    if (warp * S >= P.n_sites) return;                  // warp-uniform
    uint32_t h = warp * S + (lane % S);
    const int j = lane / S;
    const bool live = h < P.n_sites;
    if (!live) h = P.n_sites - 1u;                      // keeps the lane in the shuffles; no store
#if GF_PDL
    asm volatile("griddepcontrol.wait;" ::: "memory");
#endif
    // Run-ahead fix loop (gf_api.cu, fix_phase_runahead): the reduction that found theta below the target set this word;
    // the half-sweeps that were already enqueued behind it do nothing.  The word was written by an earlier grid of the
    // stream, which the wait above has awaited; after the first warp of an SM the load is an L1 hit.  Tested at once: a
    // value held across the solve costs the one-lane fp32 / 12-real kernel 21 registers.
#if GF_STOP_CHECK
    {
        uint32_t stopped;
        asm volatile("ld.global.ca.u32 %0, [%1];" : "=r"(stopped) : "l"(P.stop) : "memory");
        if (stopped != 0u) return;
    }
#endif
    if (P.slice_list != nullptr) {
        // frozen time slices (reading A17b) are not part of the launch at all: the grid covers the listed slices only,
        // position i of the list standing for slice slice_list[i]
        const uint32_t i = fdiv(h, G.div_sh);
        h = (uint32_t)P.slice_list[i] * G.sh + (h - i * G.sh);
    }
    const Site s = decode_site(G, h, parity);

    if (MODE == MODE_ACC && j == 0) {
        // G(x) is only needed after the links have been written back: start moving it towards L2 now
        const char* gp = link_address<T, RECON>(P.gtrans + (size_t)parity * RECON * padded_vh<T>(G), h);
        constexpr int CH = (RECON * (int)sizeof(T)) / 16;      // whole 16-byte chunks (the fp32/18 tail rides along)
#pragma unroll
        for (int c = 0; c < CH; ++c) asm volatile("prefetch.global.L2 [%0];" ::"l"(gp + (size_t)c * Tile<T>::W * 16));
    }

    // a2: gather this lane's links.  MODE_DEFER: the temporal links stay where they are; the lane that owns mu = 0
    // carries G(x) in that register slot instead (loaded up front with the links; mu = 0 does not enter K in Coulomb
    // gauge, mu0 = 1) and has no backward link there.  The lanes of a warp run the same instruction stream -- G(x) is
    // a forward link read from another base pointer, the missing backward link a masked-off load and product -- so
    // with two or four lanes per site the warp issues no more than the plain kernel does.
    T Uf[ND][18], Ub[ND][18];
    uint32_t hb[ND];
    T* const gblock = MODE == MODE_PLAIN ? nullptr : P.gtrans + (size_t)parity * RECON * padded_vh<T>(G);
    const bool gslot = MODE == MODE_DEFER && j == 0;
#pragma unroll
    for (int d = 0; d < ND; ++d) {
        const int mu = j * ND + d;
        hb[d] = backward_index(G, s, mu);
        const bool is_g = d == 0 && gslot;
        load_link<RECON>(is_g ? gblock : P.links + block_offset<T>(parity, mu, RECON, G), h, Uf[d]);
        if (is_g) {
#pragma unroll
            for (int k = 0; k < 18; ++k) Ub[d][k] = T(0);
        } else {
            // the temporal link below the first local time slice belongs to the slab below
            const T* back = (mu == 0 && s.c[0] == 0) ? P.prev_links : P.links;
            load_link<RECON>(back + block_offset<T>(parity ^ 1u, mu, RECON, G), hb[d], Ub[d]);
        }
    }
    // 12-real storage.  LAZY12: the third rows are never kept: they are formed for K(x) and dropped, and formed
    // again for the forward links in step a6 (U g^dagger does not need the third row of U at all) -- 24 flops per
    // forward link for 12 registers per link held across the solve.
    constexpr bool LAZY12 = RECON == 12 && Lazy12<T, L>::value;
    if (RECON == 12 && !LAZY12) {
#pragma unroll
        for (int d = 0; d < ND; ++d) {
            reconstruct_row2(Uf[d]);
            reconstruct_row2(Ub[d]);
        }
    }

    // a3: K(x) = sum_mu [U_mu(x) + U_mu(x-mu)^dagger]  (eq. 8, neighbours' g = 1)
    TK K[18];
#pragma unroll
    for (int k = 0; k < 18; ++k) K[k] = TK(0);
#pragma unroll
    for (int d = 0; d < ND; ++d) {
        const int mu = j * ND + d;
        if (mu >= P.mu0) {
            if (LAZY12) {
                T rf[6], rb[6];
                row2_of(Uf[d], rf);
                row2_of(Ub[d], rb);
#pragma unroll
                for (int a = 0; a < 3; ++a)
#pragma unroll
                    for (int b = 0; b < 3; ++b) {
                        const T fr = a < 2 ? GF_RE(Uf[d], a, b) : rf[2 * b], fi = a < 2 ? GF_IM(Uf[d], a, b) : rf[2 * b + 1];
                        const T br = b < 2 ? GF_RE(Ub[d], b, a) : rb[2 * a], bi = b < 2 ? GF_IM(Ub[d], b, a) : rb[2 * a + 1];
                        GF_RE(K, a, b) += (TK)fr + (TK)br;
                        GF_IM(K, a, b) += (TK)fi - (TK)bi;
                    }
            } else {
#pragma unroll
                for (int a = 0; a < 3; ++a)
#pragma unroll
                    for (int b = 0; b < 3; ++b) {
                        GF_RE(K, a, b) += (TK)GF_RE(Uf[d], a, b) + (TK)GF_RE(Ub[d], b, a);
                        GF_IM(K, a, b) += (TK)GF_IM(Uf[d], a, b) - (TK)GF_IM(Ub[d], b, a);
                    }
            }
        }
    }
#pragma unroll
    for (int off = S; off < 32; off <<= 1) {
#pragma unroll
        for (int k = 0; k < 18; ++k) K[k] += shfl_xor_T(K[k], off);
    }

    // a5: the stochastic-relaxation draws, one Philox call per site visit
    bool sq0 = false, sq1 = false, sq2 = false;
    if (P.algo == ALGO_STOCHASTIC) {
        uint32_t w[4];
        philox4x32_10(P.site_offset + 2u * h + s.xodd, 0u, counter, 0u, P.key0, P.key1, w);
        sq0 = (double)(w[0] >> 8) * (1.0 / 16777216.0) < P.p;
        sq1 = (double)(w[1] >> 8) * (1.0 / 16777216.0) < P.p;
        sq2 = (double)(w[2] >> 8) * (1.0 / 16777216.0) < P.p;
    }

    // a4: the three SU(2) subgroups, g = E3 E2 E1
    TK gk[18];
    solve_site(K, P.algo, P.omega, sq0, sq1, sq2, gk);
    T g[18];
#pragma unroll
    for (int k = 0; k < 18; ++k) g[k] = (T)gk[k];

    // a6: U_mu(x) <- g U_mu(x),  U_mu(x-mu) <- U_mu(x-mu) g^dagger  (eq. 3)
    if (!live) return;
    {
#pragma unroll
    for (int d = 0; d < ND; ++d) {
        const int mu = j * ND + d;
        const bool is_g = d == 0 && gslot;              // this slot holds G(x): G(x) <- g(x) G(x), no backward link
        T out[18];
        if (LAZY12) {                                   // the third row of the forward link again, not merged with a3's
            forget(GF_RE(Uf[d], 0, 1));
            forget(GF_RE(Uf[d], 0, 2));
            reconstruct_row2(Uf[d]);
        }
        mul_g_U<ROWS>(g, Uf[d], out);
        store_link<RECON>(is_g ? gblock : P.links + block_offset<T>(parity, mu, RECON, G), h, out);
        if (!is_g) {
            mul_U_gdag<ROWS>(Ub[d], g, out);
            T* back = (mu == 0 && s.c[0] == 0) ? P.prev_links : P.links;
            store_link<RECON>(back + block_offset<T>(parity ^ 1u, mu, RECON, G), hb[d], out);
        }
    }
    if (MODE == MODE_ACC && j == 0) {
        T* blk = gblock;
        T Gt[18], out[18];
        load_link<RECON>(blk, h, Gt);
        if (RECON == 12) reconstruct_row2(Gt);
        mul_g_U<ROWS>(g, Gt, out);
        store_link<RECON>(blk, h, out);
    }
    }
}

template <typename T, typename TK, int RECON, int L, int MODE>
__global__ void sweep_kernel(const SweepConsts<T, TK> P)
{
    sweep_body<T, TK, RECON, L, MODE>(P);
}

// The fp32 / 18-real two-lane kernels sit at 134-141 registers, just above the 128 that let 16 instead
// of 12 warps be resident; capping them (no spills with the fp32 solver) buys 3-4 % at 32^4.  Every
// other variant is better off with the allocation the compiler picks on its own, hence a second
// entry point instead of bounds on all of them.  Blocks have at most 256 threads (sweep_config_valid).
template <typename T, typename TK, int RECON, int L, int MODE>
__global__ void __launch_bounds__(256, 2) sweep_kernel_r128(const SweepConsts<T, TK> P)
{
    sweep_body<T, TK, RECON, L, MODE>(P);
}

// Only with the fp32 solver: K(x) and the SU(2) solves in fp64 registers do not fit 128 registers (the capped entry
// spilled 10 loads + 10 stores per thread), that variant takes the uncapped entry like every other.
template <typename T, typename TK, int RECON, int L> struct UseR128 {
    static constexpr bool value = sizeof(T) == 4 && sizeof(TK) == 4 && RECON == 18 && L == 2;
};

template <typename Kernel, typename Consts>
static cudaError_t launch_pdl(Kernel kernel, uint32_t grid, int block, cudaStream_t st, const Consts& P)
{
    uniform_carveout(kernel);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid, 1, 1);
    cfg.blockDim = dim3((unsigned)block, 1, 1);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = GF_PDL;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, P);
}

template <typename T, typename TK, int RECON, int L, int MODE>
static cudaError_t launch_kernel(uint32_t grid, int block, cudaStream_t st, const SweepConsts<T, TK>& P)
{
    if constexpr (UseR128<T, TK, RECON, L>::value) {
        return launch_pdl(sweep_kernel_r128<T, TK, RECON, L, MODE>, grid, block, st, P);
    } else {
        return launch_pdl(sweep_kernel<T, TK, RECON, L, MODE>, grid, block, st, P);
    }
}

template <typename T, typename TK, int RECON, int L>
static cudaError_t launch_one(int block, const SweepArgs& a, cudaStream_t st)
{
    SweepConsts<T, TK> P;
    P.links = static_cast<T*>(a.links);
    P.gtrans = static_cast<T*>(a.gtrans);
    P.slice_list = a.slice_list;
    P.n_sites = a.slice_list ? a.n_listed * a.G.sh : a.G.Vh;
    P.prev_links = a.prev_links ? static_cast<T*>(a.prev_links) : P.links;
    P.site_offset = a.site_offset;
    P.G = a.G;
    P.parity = a.parity;
    P.mu0 = a.mu0;
    P.algo = a.algo;
    P.omega = (TK)a.omega;
    P.p = a.p;
    P.key0 = a.key0;
    P.key1 = a.key1;
    P.counter = a.counter;
    P.reverse = a.reverse;
    P.stop = a.stop;
    if (P.n_sites == 0) return cudaSuccess;             // every slice frozen: nothing to launch
    const uint64_t threads = (uint64_t)P.n_sites * L;
    const uint32_t grid = (uint32_t)((threads + block - 1) / block);
    cudaError_t e;
    if (a.gtrans && a.defer_temporal)
        e = launch_kernel<T, TK, RECON, L, MODE_DEFER>(grid, block, st, P);
    else if (a.gtrans)
        e = launch_kernel<T, TK, RECON, L, MODE_ACC>(grid, block, st, P);
    else
        e = launch_kernel<T, TK, RECON, L, MODE_PLAIN>(grid, block, st, P);
    const cudaError_t sticky = cudaGetLastError();        // clears it; the launch's own code names the cause more precisely
    return e != cudaSuccess ? e : sticky;
}

bool sweep_config_valid(int lanes, int block)
{
    return (lanes == 1 || lanes == 2 || lanes == 4) && (block == 64 || block == 128 || block == 256);
}

template <typename T, typename TK, int RECON>
static cudaError_t launch_lanes(int lanes, int block, const SweepArgs& a, cudaStream_t st)
{
    switch (lanes) {
        case 1: return launch_one<T, TK, RECON, 1>(block, a, st);
        case 2: return launch_one<T, TK, RECON, 2>(block, a, st);
        case 4: return launch_one<T, TK, RECON, 4>(block, a, st);
    }
    return cudaErrorInvalidValue;
}

template <typename T, typename TK>
static cudaError_t launch_recon(int recon, int lanes, int block, const SweepArgs& a, cudaStream_t st)
{
    return recon == 12 ? launch_lanes<T, TK, 12>(lanes, block, a, st) : launch_lanes<T, TK, 18>(lanes, block, a, st);
}

cudaError_t launch_sweep(int precision, int solver_f64, int recon, int lanes, int block, const SweepArgs& a, cudaStream_t st)
{
    if (!sweep_config_valid(lanes, block)) return cudaErrorInvalidValue;
    if (precision == PREC_F64) return launch_recon<double, double>(recon, lanes, block, a, st);
    return solver_f64 ? launch_recon<float, double>(recon, lanes, block, a, st)
                      : launch_recon<float, float>(recon, lanes, block, a, st);
}

}  // namespace gf
