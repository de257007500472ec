/*
 * gf.h -- C ABI of libgf_b200: SU(3) lattice gauge fixing by checkerboard relaxation on one
 * NVIDIA B200 (sm_100a).
 *
 * The problem the calls follow (Schroeck & Vogt, arXiv:1305.3440; PAPER.md = its text):
 * given links U_mu(x) in SU(3) on a periodic N_t x N_x x N_y x N_z lattice, find the gauge
 * transformation g(x) that makes the functional F^g[U] (eq. 2) stationary, by
 * sweeping over the two parity sublattices and replacing, at every site, the links
 * by  g(x) U_mu(x)  and  U_mu(x-mu) g(x)^dagger  (eq. 3) with g(x) the local
 * maximiser of Re tr[g(x) K(x)] (eq. 7-9), until the precision theta
 * (eq. 4-5) falls below a target.
 *
 * Conventions
 *   dims[4] = {N_t, N_x, N_y, N_z}, every extent even and >= 2, N_t <= 4096.
 *   mu = 0 is time, mu = 1,2,3 = x,y,z.  parity(x) = (t+x+y+z) mod 2.
 *   Canonical link layout (what callers hold): contiguous complex array of shape
 *   (N_t, N_z, N_y, N_x, 4, 3, 3): site s = x + N_x (y + N_y (z + N_z t)), then mu, then the
 *   3x3 matrix row-major, (re, im) interleaved; complex128 or complex64.
 *   The internal device layout (parity-split, tiles of 32 / 64 sites stored as 16-byte chunks, 18 or
 *   12 reals per link) is private; gf_pack / gf_unpack convert.
 *
 * Memory and streams
 *   Every DEVICE buffer (link storage, workspace, canonical staging) is allocated by the caller
 *   (e.g. a torch tensor's data_ptr()), must be 16-byte aligned, and is only borrowed by the
 *   context until gf_destroy.  The library allocates no device memory (only a few KB of pinned
 *   host memory for scalar results), launches work only on the stream given to gf_init_lattice,
 *   and never synchronises the device except where stated.  Pointers named dev_* are device
 *   pointers, host_* are host pointers.
 *
 * Errors
 *   Every int-returning call returns GF_OK (0), a positive informational code with valid
 *   outputs, or a negative error; nothing throws, aborts or prints.  gf_last_error gives the
 *   text of the last error of a context.  Argument errors are detected before any launch, so a
 *   call that fails with GF_EINVAL / GF_ESTATE leaves the link field unchanged.
 */
#ifndef GF_B200_H
#define GF_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gf_ctx gf_ctx; /* opaque; owned by the library; freed by gf_destroy */

enum { GF_OK = 0, GF_NOT_CONVERGED = 1, GF_EINVAL = -1, GF_ENOMEM = -2, GF_ECUDA = -3, GF_ESTATE = -4 };
enum { GF_LANDAU = 0, GF_COULOMB = 1 };                   /* gauge */
enum { GF_F32 = 0, GF_F64 = 1, GF_MIXED = 2, GF_MIXED_EXACT = 3 }; /* precision */
enum { GF_RELAX = 0, GF_OVERRELAX = 1, GF_STOCHASTIC = 2 }; /* algo: PAPER.md:73, :80, :84 */
enum { GF_RECON18 = 18, GF_RECON12 = 12 };                /* reals stored per link */

/* Bytes of device memory one internal link field needs: 8 * ceil(V/2 to whole layout tiles) * recon * sizeof(real)
 * (tiles of 32 sites in fp64, 64 in fp32: exactly V * 4 * recon * sizeof(real) when V/2 is a multiple of that).
 * precision is GF_F32 or GF_F64.  Returns 0 for invalid arguments. */
size_t gf_storage_bytes(const int dims[4], int precision, int recon);

/* Bytes of device scratch the reductions need (per-block partial sums).  0 if dims invalid. */
size_t gf_workspace_bytes(const int dims[4]);

/* Creates a context.  gauge: GF_LANDAU (K, F, theta over mu = 0..3) or
 * GF_COULOMB (over the spatial mu = 1..3, F and theta per time slice; the transformation still
 * acts on all eight links of a site).  recon: GF_RECON18 stores all 9 complex entries,
 * GF_RECON12 stores rows 0 and 1 and rebuilds row 2 = conj(row0 x row1) on load.
 * dev_links_f64 / dev_links_f32: storage of gf_storage_bytes() each, either may be NULL if that
 * precision is never used (GF_MIXED needs both).  dev_workspace: gf_workspace_bytes().
 * cuda_stream: a cudaStream_t (NULL = the legacy default stream).  seed: key of the Philox
 * generator used by GF_STOCHASTIC; the half-sweep counter starts at 0.
 * Errors: GF_EINVAL (bad dims / enum / alignment / both link pointers NULL), GF_ENOMEM,
 * GF_ECUDA (no sm_100 device, ...; *out is then NULL). */
int gf_init_lattice(gf_ctx** out, const int dims[4], int gauge, int recon, void* dev_links_f64,
                    void* dev_links_f32, void* dev_workspace, void* cuda_stream, uint64_t seed);

/* canonical (device) -> internal field of `precision` (GF_F32 | GF_F64); converts the real type
 * if canonical_is_f64 differs.  Asynchronous on the context's stream.  The canonical buffer (here and in gf_unpack,
 * gf_transform_pack / _unpack; the staging buffer of gf_load_host / gf_store_host) is moved as 16-byte vectors:
 * a pointer that is not 16-byte aligned is refused with GF_EINVAL. */
int gf_pack(gf_ctx* ctx, const void* dev_canonical, int canonical_is_f64, int precision);

/* internal field of `precision` -> canonical (device); GF_RECON12 rebuilds row 2.  Asynchronous. */
int gf_unpack(gf_ctx* ctx, void* dev_canonical, int canonical_is_f64, int precision);

/* Host-buffer variants: copy a canonical field between HOST memory (pinned for a truly
 * asynchronous copy) and the internal field, staging through dev_staging (a caller-owned device
 * buffer of V*4*9*2*sizeof(real of the canonical type) bytes).  gf_load_host is asynchronous;
 * gf_store_host synchronises the stream before returning, so host_canonical is complete. */
int gf_load_host(gf_ctx* ctx, const void* host_canonical, int canonical_is_f64, int precision,
                 void* dev_staging);
int gf_store_host(gf_ctx* ctx, void* host_canonical, int canonical_is_f64, int precision,
                  void* dev_staging);

/* One half-sweep: every site x of `parity` (0|1) forms
 * K(x) = sum_mu [U_mu(x) + U_mu(x-mu)^dagger] (eq. 8, neighbours' g = 1), runs the three SU(2)
 * subgroup maximisations (0,1), (0,2), (1,2) (eq. 9 on the SU(2) projection of each 2x2 block,
 * K refreshed in between), modified per `algo`: GF_RELAX as is; GF_OVERRELAX a -> normalise(1 +
 * omega (a - 1)), omega in [1,2); GF_STOCHASTIC a -> a^2 if u < p, p in [0,1], u the
 * Philox4x32-10 draw of (seed; site, half-sweep counter; subgroup); then writes
 * g U_mu(x) and U_mu(x-mu) g^dagger in place (eq. 3).  precision: GF_F32 | GF_F64 selects the
 * field and the arithmetic.  Enqueues one kernel and returns without synchronising; increments
 * the context's half-sweep counter.  Errors: GF_EINVAL (parity, algo, omega, p, precision),
 * GF_ESTATE (no storage for that precision), GF_ECUDA. */
int gf_sweep(gf_ctx* ctx, int parity, int algo, double omega, double p, int precision);

/* n iterations = n x {gf_sweep(parity 0); gf_sweep(parity 1)}, enqueued without synchronising; the
 * Philox counter advances by 2 per iteration.  (A fused both-parities launch in t-wavefront order was built and
 * measured in rounds 1 and 2 and removed: it did not beat two half-sweeps on B200.)
 * Errors: as gf_sweep. */
int gf_iterate(gf_ctx* ctx, int n, int algo, double omega, double p, int precision);

/* F (eq. 2) and theta (eq. 4-5, with A_mu the traceless
 * anti-Hermitian part of U_mu) of the field of `precision`, accumulated in fp64 with a fixed
 * reduction order.  host_out receives 1 double (Landau) or N_t doubles (Coulomb: per time slice,
 * spatial directions, normalised by N_s^3).  These calls synchronise the stream.
 * gf_measure computes both in one pass over the field; either pointer may be NULL. */
int gf_functional(gf_ctx* ctx, int precision, double* host_out);
int gf_theta(gf_ctx* ctx, int precision, double* host_out);
int gf_measure(gf_ctx* ctx, int precision, double* host_functional, double* host_theta);

/* The same reduction without stalling the stream: gf_measure_async enqueues the F / theta pass over the
 * field as it is at that point of the stream; the kernels write the per-slice sums straight into
 * pinned host memory, slot 0..15.  gf_measure_collect synchronises the stream and returns the values
 * of a slot exactly as gf_measure would have (either pointer may be NULL), then frees the slot.
 * For following the convergence of a run without a host round trip per evaluation.
 * Errors: GF_EINVAL (slot), GF_ESTATE (empty slot, no storage), GF_ECUDA. */
int gf_measure_async(gf_ctx* ctx, int precision, int slot);
int gf_measure_collect(gf_ctx* ctx, int slot, double* host_functional, double* host_theta);

/* ---- F and theta for callers that cannot allocate.
 * Every other call needs a gf_ctx, and gf_init_lattice allocates (the context on the heap, pinned host memory,
 * events) and is handed a workspace the caller had to allocate.  Some callers can do neither at the point where they
 * want theta: a monitor hooked into another program's update loop once that program's pool allocator owns all of the
 * GPU's memory (cudaMalloc then fails and the pool is not yours to ask), a job whose memory budget is fixed and checked
 * at start-up, a latency-bound loop that cannot afford the device-wide synchronisation that cudaMalloc,
 * cudaMallocHost and cudaFree bring with them.  gf_measure_static is for them: it calls no cudaMalloc / cudaFree /
 * cudaMallocHost and no library routine that allocates, creates no context, and takes only inputs and outputs.
 *
 * What it computes: exactly what gf_measure computes (PAPER.md:39 eq. 2, :50-52 eq. 4-5; same kernels, same summation
 * order, bitwise the same numbers) for the lattice `dims`, `gauge`, and the INTERNAL link field dev_links of
 * `precision` (GF_F32 | GF_F64) and `recon` -- the buffer gf_pack / gf_sweep of a context with the same dims,
 * precision and recon wrote (gf_storage_bytes, 16-byte aligned), treated as periodic (no slabs).  dev_links is only read.
 * dev_out (DEVICE pointer, 8-byte aligned; mapped pinned host memory works too) receives, for GF_LANDAU, 2 doubles
 * {F, theta}; for GF_COULOMB 2 N_t doubles {F_t, theta_t} for t = 0 .. N_t-1, interleaved.  Asynchronous on
 * cuda_stream (a cudaStream_t of the CURRENT device, which must be the one holding dev_links and dev_out; NULL = the
 * legacy default stream); the values are there once the stream has reached this point.
 *
 * Scratch: the partial sums between the two reduction kernels live in an array that is part of the library's device
 * image, 1 114 368 bytes on every GPU that loads the library, held until the process exits.  Hence
 *   - the limit: N_t * 2 * ceil(N_x N_y N_z / 256) <= GF_STATIC_MAX_BLOCKS (up to 8.4 M sites: 32^4, 48^4, 64^3 x 32,
 *     32^3 x 64 fit; 64^4 does not).  Larger lattices are refused with GF_EINVAL before anything is launched;
 *   - every call on a device uses the same array and finds what the last call left; the call clears the one word that
 *     has to start at zero itself.  Two calls that OVERLAP on the GPU (different streams without an ordering between
 *     them, or several host threads) race on it and both results are then garbage: order them (same stream, or events);
 *   - the first call on each device looks up the array's device address (cudaGetSymbolAddress) and checks the device's
 *     architecture; later calls only launch.  Make that first call during set-up, before any stream capture begins.
 * Errors: GF_EINVAL (dims, enums, NULL or misaligned pointers, lattice beyond the limit) and GF_ECUDA for a device
 * that is not sm_100, both found before anything is launched; GF_ECUDA for a failed launch.  There is no context to keep
 * an error text: host_err (HOST buffer of host_err_len bytes, may be NULL / 0) receives it, NUL-terminated, "" on success. */
enum { GF_STATIC_MAX_BLOCKS = 65536 };
int gf_measure_static(const int dims[4], int gauge, int precision, int recon, const void* dev_links,
                      double* dev_out, void* cuda_stream, char* host_err, size_t host_err_len);

/* Iterates {gf_sweep(parity 0); gf_sweep(parity 1)} (= 1 iteration); after every
 * iteration that is a multiple of check_every (and after the last) evaluates theta (Coulomb:
 * max over slices) and stops when it is below theta_target.  precision GF_MIXED: fp32
 * iterations until theta < max(theta_target, 1e-6), then gf_cast fp32->fp64 (with SU(3)
 * re-projection) and fp64 iterations; the fp32 field must hold the input and the result is in
 * the fp64 field.  precision GF_MIXED_EXACT (needs both link fields and both transformation
 * buffers): the fp64 field holds the input and is not rounded; it is copied to fp32, fp32
 * iterations record G(x) from the identity until theta < max(theta_target, 1e-6), then the
 * untouched fp64 input is transformed by the re-projected G (gf_transform_cast +
 * gf_apply_transform), and fp64 iterations continue, accumulating into the fp64 transformation:
 * the result equals G(x) U_mu(x) G(x+mu)^dagger of the input to fp64 accuracy and G is returned
 * in the fp64 transformation buffer.  *iters_out = iterations done (both phases), *theta_out = last theta;
 * with GF_MIXED / GF_MIXED_EXACT theta is always (re-)measured on the fp64 result, also when the fp32 phase
 * already met the target or used up max_iter.
 * Returns GF_OK, or GF_NOT_CONVERGED (valid outputs) when max_iter was reached.  Synchronises. */
int gf_fix_until(gf_ctx* ctx, int algo, double omega, double p, int precision, double theta_target,
                 int max_iter, int check_every, int* iters_out, double* theta_out);

/* ---- The accumulated gauge transformation G(x) (eq. 3).
 * A relaxation sweep replaces the links by g(x) U_mu(x) g(x+mu)^dagger site after site; the
 * product of all g(x) applied to a site so far, G(x), is what a user needs to transform other
 * fields, and what lets a low-precision run be replayed on the untouched input.
 *
 * gf_transform_bytes: device bytes of one transformation field (one 3x3 matrix per site, stored
 * like a link with `recon` reals) = gf_storage_bytes / 4.
 * gf_set_transform: lends the context one buffer per precision (either may be NULL; both NULL
 * detaches).  While a buffer for precision P is attached, every gf_sweep / gf_fix_until sweep of
 * precision P also does G(x) <- g(x) G(x) on the sites it visits (one more matrix read and
 * written per site-update: +12.5 % memory traffic).  Attaching does not initialise the buffer.
 * gf_transform_identity: G(x) = 1.  gf_transform_pack / gf_transform_unpack: canonical (device)
 * <-> internal; canonical = contiguous complex array (N_t, N_z, N_y, N_x, 3, 3), complex128 or
 * complex64.  gf_transform_cast: copies G between the precisions; fp32 -> fp64 re-projects every
 * matrix onto SU(3) (Gram-Schmidt) in fp64.  All asynchronous on the context's stream.
 * Errors: GF_EINVAL (alignment, enum, null pointer), GF_ESTATE (no buffer for that precision). */
size_t gf_transform_bytes(const int dims[4], int precision, int recon);
int gf_set_transform(gf_ctx* ctx, void* dev_g_f64, void* dev_g_f32);
int gf_transform_identity(gf_ctx* ctx, int precision);
int gf_transform_pack(gf_ctx* ctx, const void* dev_canonical, int canonical_is_f64, int precision);
int gf_transform_unpack(gf_ctx* ctx, void* dev_canonical, int canonical_is_f64, int precision);
int gf_transform_cast(gf_ctx* ctx, int from_precision, int to_precision);

/* Link field of dst_precision <- G(x) U_mu(x) G(x+mu)^dagger of the link field of src_precision
 * (eq. 3), with G the transformation of g_precision.  The products are formed in fp64 whatever
 * the storage; an fp32 G is re-projected onto SU(3) in fp64 first, so the result is gauge
 * equivalent to the source to fp64 accuracy.  src_precision == dst_precision works in place.
 * Asynchronous.  Errors as above. */
int gf_apply_transform(gf_ctx* ctx, int g_precision, int src_precision, int dst_precision);

/* ---- Coulomb-gauge specialisation (the paper only names Coulomb gauge,
 * PAPER.md:11, :29).  In Coulomb gauge K(x), F_t and theta_t involve the spatial links only, and
 * the spatial links of time slice t are changed only by the sites of slice t: the slices are
 * independent problems.  Two options follow, both off by default, GF_COULOMB contexts only:
 *
 * defer_temporal = 1: a sweep leaves the temporal links U_0 alone and records the transformation
 *   instead, G(x) <- g(x) G(x) in the transformation buffer of the swept precision (which must be
 *   attached with gf_set_transform and is restarted from the identity by the first such sweep):
 *   6 links + G instead of 8 links are read and written per site-update (-12.5 % traffic).
 *   gf_coulomb_finish(precision) then applies U_0(x) <- G(x) U_0(x) G(x+0)^dagger (eq. 3) once,
 *   after which the field is what the plain sweeps would have produced (up to rounding order).
 *   gf_fix_until finishes by itself; gf_unpack, gf_store_host, gf_cast, gf_plaquette,
 *   gf_unitarity, gf_reunitarize and gf_apply_transform finish a pending update first; gf_pack
 *   discards it.  F and theta do not depend on the temporal links.
 * freeze_slices = 1: gf_fix_until stops sweeping a time slice once its theta_t is below the
 *   target at an evaluation (reading A17b); it returns when all slices are frozen.
 *   Every slice ends exactly where the unfrozen run has it at that iteration; the later sweeps of
 *   the unfrozen run (which keep lowering theta_t of the early slices) are saved.
 *
 * gf_set_slice_mask: explicit control for gf_sweep: host_active[t] != 0 means the sites of slice t
 * are visited (N_t bytes, HOST pointer, copied before returning); NULL = all slices.  gf_fix_until
 * with freeze_slices manages the mask itself and leaves it off.  The library turns the mask into the
 * list of active slices and a half-sweep is launched over the sites of those slices only, so slices
 * that converge at different times cost nothing once frozen (the time of a half-sweep is proportional
 * to the number of active slices); with no active slice nothing is launched.
 * While a deferred update is outstanding the transformation buffer of that precision holds the only copy of
 * what still has to be applied to U_0: gf_transform_identity, gf_transform_pack, gf_transform_cast INTO it and
 * gf_set_transform replacing it return GF_ESTATE until gf_coulomb_finish (or a call that finishes implicitly)
 * has run; gf_apply_transform / gf_cast into ANOTHER precision's field drop that field's own outstanding update
 * (the field is overwritten).
 * Errors: GF_EINVAL (Landau context, bad flag), GF_ESTATE (no transformation buffer). */
int gf_set_coulomb_mode(gf_ctx* ctx, int defer_temporal, int freeze_slices);
int gf_coulomb_finish(gf_ctx* ctx, int precision);
int gf_set_slice_mask(gf_ctx* ctx, const uint8_t* host_active);

/* ---- Slab decomposition along t (the paper's multi-GPU scheme, PAPER.md:98-117,
 * re-done over peer memory).  A lattice of nranks * N_t time slices is cut into nranks slabs of N_t
 * slices, one context (one GPU) each; dims given to gf_init_lattice are the LOCAL ones.  The only
 * data a slab shares with a neighbour are the temporal links U_0 of its last slice: the sites of the
 * first slice of the slab above read and write them IN PLACE through dev_prev_links_* (a pointer
 * into the neighbour's link field: a peer mapping over NVLink, CUDA IPC between processes, or plain
 * device memory when several slabs live on one GPU) -- no halo buffers, no exchange step, no
 * collective.  dev_next_links_* is read by gf_plaquette only.
 *
 * Ordering: every link operation (gf_pack, gf_unpack, gf_sweep, gf_measure/gf_functional/gf_theta,
 * gf_plaquette, gf_unitarity, gf_reunitarize, gf_cast) is numbered per slab; operation n of a slab
 * starts when both neighbours have completed their operation n-1.  Completion counts live in one
 * 32-bit device word per slab (dev_flag_*, zero-initialised by the caller, 4-byte aligned, the
 * neighbours' words mapped like their fields) and are written and awaited with stream memory
 * operations (cuStreamWriteValue32 / cuStreamWaitValue32): no kernel spins, the host never blocks.
 * ALL SLABS MUST ISSUE THE SAME SEQUENCE OF OPERATIONS.
 *
 * Results: links are those of the undivided lattice (sweep-by-sweep parity with the oracle; Philox
 * uses the global site index).  Landau gf_measure / gf_functional / gf_theta / gf_plaquette return
 * this slab's SHARE of the global value (local sum over the global normalisation): the caller adds
 * the slabs up (one scalar all-reduce).  Coulomb values are per local time slice.  Not available on
 * slabs (GF_ESTATE): gf_fix_until (the caller iterates and reduces theta), the transformation field,
 * deferred temporal links.  nranks = 1 restores the single-lattice behaviour.
 * Errors: GF_EINVAL (rank, missing pointers, alignment, global volume >= 2^32), GF_ESTATE, GF_ECUDA. */
int gf_set_slab(gf_ctx* ctx, int rank, int nranks, void* dev_prev_links_f64, void* dev_prev_links_f32,
                void* dev_next_links_f64, void* dev_next_links_f32, uint32_t* dev_flag_own,
                uint32_t* dev_flag_prev, uint32_t* dev_flag_next);

/* Devices.  A context belongs to the CUDA device that was current in gf_init_lattice (the one its buffers and
 * stream live on); every call makes that device current for its duration and restores the caller's, so one
 * process may drive contexts on several GPUs.  gf_get_device returns it.  gf_enable_peer(ctx, peer_device):
 * enables peer access from the context's device to peer_device (no-op for the same device or when already
 * enabled) -- needed before gf_set_slab is given pointers into a field on another GPU of the same process.
 * Errors: GF_EINVAL (no such device), GF_ECUDA (the two devices are not peers).  Multi-GPU slabs have not run
 * on hardware in this repository's pool (one GPU); see DESIGN.md section 12. */
int gf_enable_peer(gf_ctx* ctx, int peer_device);
int gf_get_device(const gf_ctx* ctx, int* device_out);

/* Sets the Philox key and the half-sweep counter (checkpoint/resume: the RNG state is just these). */
int gf_set_rng(gf_ctx* ctx, uint64_t seed, uint32_t half_sweep_counter);
int gf_get_counter(const gf_ctx* ctx, uint32_t* half_sweep_counter_out);

/* Re-projects every link of the field onto SU(3) (Gram-Schmidt on rows 0,1; row 2 = conj cross). */
int gf_reunitarize(gf_ctx* ctx, int precision);

/* Copies the internal field of one precision into the other; fp32 -> fp64 also re-projects. */
int gf_cast(gf_ctx* ctx, int from_precision, int to_precision);

/* Diagnostics (synchronise).  gf_plaquette: mean plaquette 1/(6 N_c V) sum Re tr[U_mu(x)
 * U_nu(x+mu) U_mu(x+nu)^dagger U_nu(x)^dagger], gauge invariant.  gf_unitarity: host_out[0] =
 * max |U U^dagger - 1| entry, host_out[1] = max |det U - 1| over all links. */
int gf_plaquette(gf_ctx* ctx, int precision, double* host_out);
int gf_unitarity(gf_ctx* ctx, int precision, double* host_out2);

/* Kernel configuration of gf_sweep for `precision`: lanes_per_site in {1,2,4} threads cooperate
 * on one site (each owns 8/lanes links; K is combined with warp shuffles); block_threads in
 * {64,128,256}.  0 = the built-in choice for the variant (storage precision, recon, solver
 * precision), measured on B200.  Results do not depend on it beyond the summation order inside K. */
int gf_set_tuning(gf_ctx* ctx, int precision, int lanes_per_site, int block_threads);

/* Mixed precision (GF_MIXED, GF_MIXED_EXACT): the fp32 phase of gf_fix_until runs until
 * theta < max(theta_target, theta_handoff).  Default 1e-6 (BASELINE.json configs[2]).  fp32 sweeps
 * keep lowering theta down to about 1e-11 (measured at 32^4), so with GF_MIXED_EXACT, whose result
 * does not inherit the fp32 rounding, a later hand-off moves most of the run to the cheaper sweeps.
 * A hand-off below what fp32 can reach makes the fp32 phase run to max_iter. */
int gf_set_mixed_handoff(gf_ctx* ctx, double theta_handoff);

/* Second hand-off criterion of the mixed-precision runs: how far fp32 sweeps can lower theta depends on the lattice
 * and the field (about 3e-12 on the 32^4 bench field), so a fixed theta_handoff is either too cautious or never
 * reached.  ratio in (0, 1]: the fp32 phase also ends at the first evaluation whose theta is not below
 * ratio x (theta of the previous evaluation), i.e. when fp32 has stopped lowering it at the rate asked for (a theta
 * that repeats bit for bit, the fixed point a deterministic run can reach at the rounding floor, counts as stalled); with
 * a small theta_handoff (e.g. 1e-15) the fp32 phase then runs exactly as long as it pays.  0 (default) = off.
 * An early hand-off costs time only: the fp64 phase always finishes the run.  Errors: GF_EINVAL. */
int gf_set_mixed_stall(gf_ctx* ctx, double ratio);

/* Order in which the blocks of consecutive gf_sweep launches walk the lattice: 1 (default) =
 * zigzag, every other half-sweep runs from the last site to the first, so that a launch starts on
 * the links the previous one touched last and finds them in the L2 cache; 0 = always ascending.
 * The links produced are bitwise the same (sites of one parity are independent). */
int gf_set_traversal(gf_ctx* ctx, int zigzag);

/* Re-projection onto SU(3) inside gf_fix_until.  The paper does not mention one (reading A16) and in fp64 none is
 * needed (|U U^dagger - 1| = 6e-13 after 20 000 iterations of a hot 32^4 field), but fp32 links lose unitarity linearly
 * with the number of site updates (8e-4 after 5 000 iterations of the same field, and F then starts to fall).
 * iterations > 0: at every evaluation point of gf_fix_until at which at least that many iterations have passed since the
 * last re-projection, the field being swept -- and the transformation recorded with it (GF_MIXED_EXACT, deferred temporal
 * links) -- is re-projected (Gram-Schmidt on rows 0 and 1 in fp64, row 2 = conj(row0 x row1)) before theta is measured.
 * 0 (default) = never: runs are then sweep by sweep those of the oracle.  Errors: GF_EINVAL. */
int gf_set_reunitarize_every(gf_ctx* ctx, int iterations);

/* How gf_fix_until follows theta ("iterated until the requested gauge precision theta has
 * been reached").  blocks = 0: after every evaluation the host waits for theta before it enqueues the
 * next check_every iterations.  blocks = 1..8 (default 4): up to that many blocks of {iterations;
 * F / theta reduction} are enqueued ahead of the one whose result the host waits for; the last
 * reduction kernel compares theta (Coulomb gauge: every theta_t) with theta_target on the device and,
 * once it is below, the half-sweeps already enqueued behind it leave the field alone.  Links,
 * iteration count, theta and the Philox stream are exactly those of blocks = 0; the GPU never idles
 * for a host round trip.  With Coulomb slice freezing (gf_set_coulomb_mode) the loop always waits,
 * because the list of active slices changes between evaluations.  Errors: GF_EINVAL. */
int gf_set_fix_runahead(gf_ctx* ctx, int blocks);

/* Arithmetic of the per-site solver when the STORAGE is fp32 (gf_sweep with GF_F32): K(x) is
 * accumulated and the three SU(2) solves run in solver_precision: GF_F64 (fp64 registers: no extra memory traffic;
 * the links stay within 1e-5 of an fp64 computation on the same input over a whole iteration at 32^4, measured
 * 2.2e-6), GF_F32 (everything in fp32: 10 % (18-real) to 20 % (12-real) faster at 32^4, but the fp32 rounding of K is
 * amplified by |K| / |v| at sites whose SU(2) projection |v| is small -- one site in 5 x 10^5 of a 32^4 field ends
 * 1.08e-5 away after one iteration, 1.4e-5 with GF_STOCHASTIC, whose g -> g^2 step doubles the amplification), or
 * GF_SOLVER_AUTO (the default) = GF_F64.  Callers that only precondition with fp32 sweeps may prefer GF_F32.
 * The 3x3 products g U and U g^dagger are always formed in the storage precision.  No effect on
 * GF_F64 sweeps. */
enum { GF_SOLVER_AUTO = -1 };
int gf_set_solver_precision(gf_ctx* ctx, int solver_precision);

/* Runs the device Philox4x32-10 on n (counter, key) pairs: dev_counters n*4, dev_keys n*2,
 * dev_out n*4 uint32 words (device pointers).  For known-answer tests.  Asynchronous. */
int gf_debug_philox(gf_ctx* ctx, int n, const uint32_t* dev_counters, const uint32_t* dev_keys,
                    uint32_t* dev_out);

/* Number of kernels this context has launched so far (for launch accounting in benchmarks). */
int gf_launch_count(const gf_ctx* ctx, uint64_t* count_out);

const char* gf_last_error(const gf_ctx* ctx);
void gf_destroy(gf_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* GF_B200_H */
