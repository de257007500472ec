// gf_internal.h -- host-side declarations shared by the translation units of libgf_b200.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "gf_device.cuh"

namespace gf {

enum { PREC_F32 = 0, PREC_F64 = 1 };

struct SweepArgs {
    void* links;            // internal field of the chosen precision
    void* gtrans;           // accumulated transformation of the same precision, or NULL
    int defer_temporal;     // Coulomb: with gtrans, leave the temporal links to gf_coulomb_finish
    const uint16_t* slice_list;    // Coulomb slice freezing: the time slices still being swept, ascending; NULL = all
    uint32_t n_listed;             // entries of slice_list
    void* prev_links;       // slab below (same precision and layout), or NULL = this field (periodic)
    uint32_t site_offset;   // global site index of the slab's first site
    Geom G;
    uint32_t parity;        // active parity
    int mu0;                // first direction entering K: 0 Landau, 1 Coulomb
    int algo;               // ALGO_*
    double omega, p;
    uint32_t key0, key1;    // Philox key = seed
    uint32_t counter;       // half-sweep counter (Philox counter word 2)
    uint32_t reverse;       // traverse the lattice backwards (L2 reuse between consecutive launches)
    const uint32_t* stop;   // device word, never NULL: non-zero = the run-ahead fix loop has reached its target on the
                            // device and this half-sweep, enqueued before the host knew, must leave the field alone
};

struct MeasureGrid {
    uint32_t Sh;            // sites per time slice per parity
    uint32_t bpp;           // blocks per (slice, parity)
    uint32_t block;         // threads per block
    const uint16_t* slice_list;   // measure only these time slices (the others keep their previous results); NULL = all
    uint32_t n_listed;
};

// last stage of a reduction (gf_aux.cu, reduce_slices_kernel)
struct ReduceTail {
    double* slice_tmp;      // 2 * N_t doubles of workspace
    uint32_t* counter;      // device word, zero between launches
    int combine;            // 0: one (scaled) pair per time slice; 1: one pair for the whole lattice in out[0], out[1]
    double scale0, scale1;  // normalisations applied to the two sums on the device
    uint32_t* stop;         // run-ahead fix loop: set *stop = 1 when theta (Coulomb: every theta_t) < target; NULL = no decision
    double target;
    // stall > 0 (fp32 phase of the mixed-precision runs): also stop when theta >= stall * (theta of the previous
    // evaluation), i.e. when fp32 no longer lowers it; *prev holds the previous value (0 = none yet)
    double stall;
    double* prev;
};

// All kernels of the library ask for the same shared-memory carveout (a hint).  The pack / unpack kernels need a few
// KB of shared memory per block, the sweep kernels none; blocks of kernels with different carveouts do not share an
// SM, so with several lattices in flight (one stream each) a conversion kernel would otherwise force SMs to drain and
// switch configuration in the middle of the other lattices' sweeps.
constexpr int kCarveoutPercent = 25;
template <typename Kernel>
inline void uniform_carveout(Kernel kernel)
{
    // cudaFuncSetAttribute acts on the CURRENT device only: one bit per device ordinal and kernel instantiation, so that
    // every GPU of a multi-device process (slabs.SlabSet) gets the hint, not just the first one used.  A benign race at
    // worst sets an attribute twice.
    static uint64_t done = 0;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return;
    const uint64_t bit = uint64_t(1) << (dev & 63);
    if (!(done & bit)) {
        cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, kCarveoutPercent);
        done |= bit;
    }
}

// Geometry and measurement grid of a lattice from its extents alone, for entry points that work without a context
// (gf_static.cu).  Must describe the lattice exactly as gf_init_lattice does: tests/test_zz_no_alloc.py compares the two.
constexpr uint32_t kMeasureBlockThreads = 128;

inline Geom make_geom(const int dims[4])
{
    Geom G;
    G.nt = (uint32_t)dims[0];
    G.nxh = (uint32_t)dims[1] / 2u;
    G.ny = (uint32_t)dims[2];
    G.nz = (uint32_t)dims[3];
    G.Vh = (uint32_t)((uint64_t)dims[0] * dims[1] * dims[2] * dims[3] / 2u);
    G.Vp[PREC_F32] = (G.Vh + Tile<float>::W - 1u) / Tile<float>::W * Tile<float>::W;
    G.Vp[PREC_F64] = (G.Vh + Tile<double>::W - 1u) / Tile<double>::W * Tile<double>::W;
    for (int mu = 0; mu < 4; ++mu) G.extent[mu] = (uint32_t)dims[mu];
    G.stride[1] = 1;
    G.stride[2] = G.nxh;
    G.stride[3] = G.nxh * G.ny;
    G.stride[0] = G.nxh * G.ny * G.nz;
    G.div_nxh = make_fastdiv(G.nxh);
    G.div_ny = make_fastdiv(G.ny);
    G.div_nz = make_fastdiv(G.nz);
    G.sh = G.Vh / G.nt;
    G.div_sh = make_fastdiv(G.sh);
    return G;
}

inline MeasureGrid make_measure_grid(const int dims[4])
{
    MeasureGrid mg;
    mg.Sh = (uint32_t)((uint64_t)dims[1] * dims[2] * dims[3] / 2u);
    mg.block = kMeasureBlockThreads;
    mg.bpp = (mg.Sh + mg.block - 1u) / mg.block;
    mg.slice_list = nullptr;
    mg.n_listed = 0;
    return mg;
}

// every launcher returns cudaGetLastError() after the launch
// solver_f64: with fp32 storage, accumulate K(x) and run the SU(2) solves in fp64 registers
cudaError_t launch_sweep(int precision, int solver_f64, int recon, int lanes, int block, const SweepArgs& a, cudaStream_t st);
bool sweep_config_valid(int lanes, int block);

// prev_links / next_links: the fields of the slabs below / above in t (NULL = this field, periodic)
cudaError_t launch_measure(int precision, int recon, const void* links, const void* prev_links, const Geom& G, int mu0,
                           const MeasureGrid& mg, double* partials, const ReduceTail& tail, double* slice_out, cudaStream_t st);
cudaError_t launch_plaquette(int precision, int recon, const void* links, const void* next_links, const Geom& G,
                             const MeasureGrid& mg, double* partials, const ReduceTail& tail, double* slice_out, cudaStream_t st);
cudaError_t launch_unitarity(int precision, int recon, const void* links, const Geom& G,
                             const MeasureGrid& mg, double* partials, const ReduceTail& tail, double* slice_out, cudaStream_t st);
cudaError_t launch_pack(int precision, int recon, void* links, const Geom& G, const void* canonical,
                        int canonical_is_f64, cudaStream_t st);
cudaError_t launch_unpack(int precision, int recon, const void* links, const Geom& G, void* canonical,
                          int canonical_is_f64, cudaStream_t st);
// nblocks: 8 for a link field (parity x mu), 2 for a transformation field (parity)
// stop: NULL, or the stop word of the run-ahead fix loop (the kernel then does nothing once it is set)
cudaError_t launch_cast(int from_precision, int to_precision, int recon, const void* src, void* dst,
                        const Geom& G, int reproject, int nblocks, cudaStream_t st, const uint32_t* stop = nullptr);
// transformation field G[parity][chunk][h] <-> canonical (V,3,3) complex; identity fill
cudaError_t launch_transform_pack(int precision, int recon, void* gtrans, const Geom& G, const void* canonical,
                                  int canonical_is_f64, cudaStream_t st);
cudaError_t launch_transform_unpack(int precision, int recon, const void* gtrans, const Geom& G, void* canonical,
                                    int canonical_is_f64, cudaStream_t st);
cudaError_t launch_transform_identity(int precision, int recon, void* gtrans, const Geom& G, cudaStream_t st);
// dst_mu(x) = G(x) src_mu(x) G(x+mu)^dagger in fp64 (eq. 3); src may alias dst
// only the directions mu_begin <= mu < mu_end are transformed
cudaError_t launch_apply_transform(int g_precision, int src_precision, int dst_precision, int recon,
                                   const void* gtrans, const void* src, void* dst, const Geom& G,
                                   int mu_begin, int mu_end, cudaStream_t st);
cudaError_t launch_philox(int n, const uint32_t* ctr, const uint32_t* key, uint32_t* out, cudaStream_t st);

}  // namespace gf
