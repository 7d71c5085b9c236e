/* =====================================================================================
 * qcd.h -- C ABI of the B200-native checkerboard SU(N) Monte Carlo sweep
 *          (hot path of QCDGPU, arxiv 1310.7087; scope table: SURVEY.md sec 8).
 *
 * What the operations are (citations: PAPER.md = the paper text; R# = reading in DESIGN.md):
 *   - links are N x N complex matrices on lattice links, N = 2,3, D = 2..4 run-time
 *     dimension, single or double precision
 *   - the lattice is updated in even/odd "checkerboard" order with a (pseudo)heat-bath,
 *     NHIT = 10 trials, followed by reunitarisation
 *   - optional external abelian (chromo)magnetic field, finite temperature
 *   - one seed reproduces a run
 *   - overrelaxation, Philox4x32-10, plaquette and Polyakov loop: BASELINE.json north_star.
 *
 * Conventions
 *   - every function returns a status code (QCD_OK = 0); nothing throws or aborts across the
 *     ABI; qcd_last_error() returns a thread-local, human-readable message for the last failure.
 *   - handles are thread-compatible, not thread-safe.
 *   - all pointers are HOST pointers unless the argument name or comment says "device".
 *   - dims[0] is the fastest axis, dims[D-1] is the time axis (Polyakov direction);
 *     every extent must be even and >= 2 (checkerboard + periodic boundary conditions).
 *   - canonical link layout (qcd_get_links / qcd_set_links): [lex site][mu][row][col][re,im]
 *     in the lattice's precision, full N x N always (SU(3): 18 reals, SU(2): 8 reals),
 *     lex = x0 + L0*(x1 + L1*(x2 + L2*x3)).
 *   - all work is enqueued on the stream given at creation; only qcd_measure, qcd_get_links
 *     (to host), the qcd_debug_get_* calls and qcd_get_profile synchronise that stream.
 * ===================================================================================== */
#ifndef QCD_B200_H
#define QCD_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct qcd_lattice qcd_lattice_t; /* opaque, library-owned */

enum { QCD_OK = 0, QCD_ERR_INVALID_ARG = 1, QCD_ERR_UNSUPPORTED = 2, QCD_ERR_ALLOC = 3, QCD_ERR_CUDA = 4, QCD_ERR_STATE = 5 };
enum { QCD_FP32 = 0, QCD_FP64 = 1 };        /* precision of storage and of the link arithmetic */
enum { QCD_FLAG_COMPRESS12 = 1u };          /* SU(3) only: store rows 0,1 (12 reals), rebuild row 2 on load */
enum { QCD_COLD = 0, QCD_HOT = 1 };
enum { QCD_KIND_HB = 0, QCD_KIND_OR = 1 };
enum {
  QCD_OPT_KP_MAX_TRIALS = 0, /* Kennedy-Pendleton trial cap, 1..127, default 10 ("NHIT=10", R5) */
  QCD_OPT_DEBUG_TRIALS = 1,  /* 1: qcd_debug_substep records per-(link,subgroup) trial codes (allocates V*3 bytes) */
  QCD_OPT_PROFILE = 2,       /* 1: CUDA events around the update kernels: one pair per run of same-kind launches in qcd_sweep,
                                one pair per launch in qcd_debug_substep (see qcd_get_profile) */
  QCD_OPT_BULK_COPY = 3,     /* 1: SU(3) fp32 x12 overrelaxation on D = 4 lattices with dims[0] = 32 runs the kernel that stages
                                every operand with bulk asynchronous copies (cp.async.bulk + mbarriers, update_bulk.cuh) instead
                                of the tiled cp.async kernel.  Same results to rounding; measured SLOWER:
                                default 0, kept so that the comparison can be repeated (bench.py --bulk-copy) */
  QCD_OPT_ALTERNATE_ORDER = 4, /* 1 (default): consecutive update launches visit the lattice in opposite directions, so that a
                                launch starts on the links the previous one touched last and finds them in the L2
                                (DESIGN.md sec 6.5).  Results are bit-identical either way; 0 restores one direction */
  QCD_OPT_EXCHANGE_ROWS01 = 5 /* 1: qcd_get_links / qcd_set_links of this lattice exchange rows 0,1 of every link only --
                                [lex site][mu][2][3][re,im], V*D*12 reals -- i.e. exactly what a 12-real (COMPRESS12) SU(3)
                                lattice stores: a third less over the host link, nothing lost (row 2 = conj(row0 x row1)).
                                SU(3) with COMPRESS12 only; default 0 (full 3 x 3) */
};

/* Constant abelian background: every plaquette of plane (mu,nu), mu < nu, is multiplied on the left, at its
 * base site, by F = diag(exp(i*theta_c)), c < N (R12).  sum_c theta_c must be 0 (|sum| <= 1e-12) so that
 * F is in SU(N).  BASELINE config 4: SU(2), plane (0,1), theta = (+phi/2, -phi/2), phi = 2*pi*n_f/(Lx*Ly). */
typedef struct {
  int enabled;
  int mu, nu;
  double theta[3];
} qcd_field_t;

/* Bytes of device workspace a lattice needs (links in the internal layout).  0 on invalid arguments and on lattices
 * beyond the kernels' indexing: V > 2^31 sites, or one (parity, direction) array of NP planes x V/2 vectors of 16 bytes
 * reaching 2^32 vectors (UNSUPPORTED; SU(3) 128^4 in fp64 x18, 154.6 GB, is within both). */
size_t qcd_lattice_bytes(int D, const int* dims, int Nc, int precision, unsigned flags);

/* Create a lattice.  device_mem: DEVICE pointer to >= qcd_lattice_bytes() bytes, 256-byte aligned, owned by the
 * caller (e.g. a torch uint8 tensor) and kept alive until qcd_lattice_destroy; NULL => the library cudaMallocs
 * and frees it.  cuda_stream: a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL => default
 * stream.  Errors: INVALID_ARG (D not in 2..4, odd/small extent, Nc not 2/3, bad precision, buffer too small
 * or misaligned), UNSUPPORTED (COMPRESS12 with Nc=2), ALLOC, CUDA. */
int qcd_lattice_create(int D, const int* dims, int Nc, int precision, unsigned flags, void* device_mem, size_t bytes,
                       void* cuda_stream, qcd_lattice_t** out);
int qcd_lattice_destroy(qcd_lattice_t* lat); /* frees only what the library allocated */

/* Set all links: QCD_COLD = identity; QCD_HOT = Haar-random SU(N) from Philox domain 1 (R9), computed in
 * double and rounded to the storage precision.  Stores the seed, sets the sweep counter to 0. */
int qcd_init(qcd_lattice_t* lat, int start, uint64_t seed);

/* One sweep (R1,R2): for pass in (n_hb heatbath hits, then n_or overrelaxation passes): for parity in (0,1):
 * for mu in 0..D-1: update every link U_mu(x), x of that parity: sum the 2(D-1) staples (with the field factor
 * when field != NULL && field->enabled), Cabibbo-Marinari update over the SU(2) subgroups (Kennedy-Pendleton
 * heatbath / overrelaxation), reunitarise, store.  Then the sweep counter is incremented.  Asynchronous.
 * Errors: STATE (no links yet), INVALID_ARG (beta not finite or < 0, n_hb/n_or < 0 or > 65535, bad field). */
int qcd_sweep(qcd_lattice_t* lat, double beta, int n_hb, int n_or, const qcd_field_t* field);

/* Observables (R10,R11): plaquette per plane = mean over sites of (1/N) Re Tr [F] U_mu(x) U_nu(x+mu) U_mu(x+nu)^+
 * U_nu(x)^+, order (0,1),(0,2),..,(D-2,D-1) (D(D-1)/2 doubles, may be NULL); plaq_total = mean over planes (may
 * be NULL); polyakov_re_im = mean over spatial sites of (1/N) Tr prod_t U_{D-1}(x,t) (2 doubles, may be NULL).
 * Site arithmetic in the lattice's precision, accumulation in fp64, deterministic.  Synchronises the stream. */
int qcd_measure(qcd_lattice_t* lat, const qcd_field_t* field, double* plaq_total, double* plaq_planes, double* polyakov_re_im);

/* Working sweep ("working sweeps" = update + measurements): qcd_sweep followed by the
 * observables of the NEW configuration, with the plaquette measurement folded into the last pass of the sweep: there the
 * sub-steps (parity 1, mu >= 1) already hold every plaquette of the planes (nu, mu), nu < mu, in its final state as
 * Re Tr[U'_mu(x) A_nu(x)], so no separate pass over the links is made for it (the Polyakov loop keeps its own small
 * kernel).  Results equal qcd_sweep + qcd_measure up to rounding (another summation order for the observables; the
 * measuring kernels are separate instantiations of the update kernels, so the links agree to a few units in the last
 * place); each call is deterministic on its own.  Arguments and errors as for those two calls; synchronises the stream.
 * n_hb + n_or = 0 measures the unchanged configuration. */
int qcd_sweep_measure(qcd_lattice_t* lat, double beta, int n_hb, int n_or, const qcd_field_t* field, double* plaq_total,
                      double* plaq_planes, double* polyakov_re_im);
/* The same with the observables added to the on-device accumulators (see below) instead of returned: asynchronous. */
int qcd_sweep_measure_accumulate(qcd_lattice_t* lat, double beta, int n_hb, int n_or, const qcd_field_t* field);

/* On-device accumulation over configurations (the paper keeps its measurements on the device until
 * the end of a run).  qcd_measure_accumulate measures like qcd_measure and adds the NQ = D(D-1)/2 + 3
 * quantities (plane plaquettes in qcd_measure's order, Re L, Im L, |L|) and their squares to accumulators in device
 * memory; it is asynchronous (no host synchronisation, nothing returned).  qcd_accum_get synchronises and returns the
 * number of accumulated measurements and the NQ sums and sums of squares (host arrays of `capacity` >= NQ doubles);
 * qcd_accum_reset zeroes the accumulators (they start at zero).  Fixed summation order: bit-reproducible. */
int qcd_measure_accumulate(qcd_lattice_t* lat, const qcd_field_t* field);
int qcd_accum_get(qcd_lattice_t* lat, uint64_t* count, double* sum, double* sumsq, int capacity);
int qcd_accum_reset(qcd_lattice_t* lat);

/* The plane plaquettes for callers that must not allocate device memory.
 *
 * Who that is: a program that has given the whole GPU to an allocator of its own -- typically a PyTorch process whose caching
 * allocator already holds nearly all of the 180 GB (a 128^4 fp64 lattice alone is 154.6 GB) -- so that a cudaMalloc made by
 * this library behind the allocator's back can fail although the pool has room, and the library cannot ask the pool (the ABI
 * carries no torch types); and a program that measures inside a steady-state loop next to other work on the same GPU (other
 * lattices on other streams), where it cannot afford cudaMalloc / cudaFree, which may stall the whole device.  qcd_measure
 * is not safe for them: when first called on a lattice it cudaMallocs its buffer of per-CTA partial sums (and creates a side
 * stream and two events).
 *
 * This call computes what qcd_measure returns in plaq_planes -- the same two kernels, launched the same way, so the numbers
 * are the same bit for bit -- but keeps the partial sums in an array built into the library's device code.  It calls no
 * cudaMalloc, cudaFree or any other allocating routine, on the first call or later.  The price: that array is
 * QCD_NOALLOC_MAX_PARTIALS doubles = 8 MiB on every GPU on which the library's device code is loaded, held until the process
 * exits whether or not this call is ever used, and it bounds the lattice: D(D-1)/2 planes x (own sites / 128, rounded up
 * per parity) partial sums must fit: in D = 4 that is 22.3 million sites (64^4 = 16.8 million fits, 128^4 does not; the 32^4
 * headline lattice uses 384 KiB of it).
 * A larger lattice is refused with QCD_ERR_UNSUPPORTED and a message naming both numbers; nothing is launched.
 *
 *   lat         an initialised lattice (not a slab); its links are the input.  Its device must be the CURRENT device.
 *   field       as for qcd_measure (NULL: none).
 *   device_out  DEVICE pointer, caller-owned, D(D-1)/2 doubles, 8-byte aligned: the plane plaquettes in qcd_measure's
 *               order (0,1),(0,2),..,(D-2,D-1); their mean is qcd_measure's plaq_total.
 * Asynchronous on the lattice's stream: device_out is valid once the work enqueued by this call has completed there.
 *
 * Set-up: the first call on each device asks the CUDA runtime for the array's address on that device
 * (cudaGetSymbolAddress; the result is cached per device).  Make that first call during set-up, before any stream capture
 * is begun in the process.
 * Sharing: there is ONE array per GPU, used by every call on every lattice and stream, and it keeps whatever the previous
 * call left in it.  That is harmless for calls that follow one another (each call overwrites every entry it later reads;
 * nothing needs to start at zero).  Two calls that can run on the GPU at the same time -- different streams, or different
 * host threads driving different lattices -- race on it and both results are garbage: order them yourself (one stream, or an
 * event between them).
 * Errors: INVALID_ARG (NULL / misaligned pointer, bad field), STATE (no links yet; lattice on another device than the
 * current one), UNSUPPORTED (slab; lattice beyond the array; device ordinal >= 64), CUDA. */
enum { QCD_NOALLOC_MAX_PARTIALS = 1 << 20 };
int qcd_measure_plaquette_noalloc(qcd_lattice_t* lat, const qcd_field_t* field, double* device_out);

/* Copy links out of / into the lattice in the canonical layout.  bytes must equal V*D*N*N*2*sizeof(real).
 * dst_is_device / src_is_device: the pointer is a DEVICE pointer, 16-byte aligned (then the call is asynchronous on the
 * stream).  HOST pointers (pageable or pinned): the transfer is staged through a bounded device buffer (64 MiB, allocated
 * on first use) in chunks of whole sites, and the call returns after the host buffer has been read / filled.
 * qcd_set_links does not reunitarise; with COMPRESS12 row 2 of the input is dropped; SU(2) input is read from
 * its first row (a0 = Re U00, a3 = Im U00, a2 = Re U01, a1 = Im U01). */
int qcd_get_links(qcd_lattice_t* lat, void* dst, size_t bytes, int dst_is_device);
int qcd_set_links(qcd_lattice_t* lat, const void* src, size_t bytes, int src_is_device);

/* Checkpoint / resume: state = canonical links + seed + sweep counter. */
int qcd_get_sweep_counter(qcd_lattice_t* lat, uint32_t* out);
int qcd_set_sweep_counter(qcd_lattice_t* lat, uint32_t value);
int qcd_get_seed(qcd_lattice_t* lat, uint64_t* out);
int qcd_set_seed(qcd_lattice_t* lat, uint64_t seed);
int qcd_set_option(qcd_lattice_t* lat, int key, int value);

/* One (parity, mu) sub-step of kind QCD_KIND_HB (heatbath hit index `hit`) or QCD_KIND_OR, with the current
 * sweep counter (not incremented).  Used by the parity tests to compare per sub-step with resync. */
int qcd_debug_substep(qcd_lattice_t* lat, double beta, int kind, int hit, int parity, int mu, const qcd_field_t* field);

/* Trial codes of the last heatbath qcd_debug_substep, [lex site][subgroup 0..2] (V*3 bytes, host): 0 = subgroup
 * skipped (k^2 tiny, R4) or site not updated; t+1 = accepted at trial t; 0x80|T_max = all trials failed (R5).
 * Needs QCD_OPT_DEBUG_TRIALS = 1. */
int qcd_debug_get_trials(qcd_lattice_t* lat, uint8_t* dst, size_t bytes);

/* Philox4x32-10 on the device for n (counter, key) pairs (host arrays: ctr 4n words, key 2n words, out 4n words).
 * impl 0: this library's generator; impl 1: cuRAND's curand_Philox4x32_10 compiled into a kernel (cross-check). */
int qcd_debug_philox(const uint32_t* ctr, const uint32_t* key, size_t n, uint32_t* out, int impl);

/* The fp64 heatbath's elementary functions (csrc/hb_math.cuh) evaluated on the device for n 32-bit words w (host arrays):
 * out[7 i + 0..6] = ln u, cos^2(2 pi u), sin(2 pi u), cos(2 pi u) with u = (w + 1/2) 2^-32, and sqrt(x), 1/sqrt(x), 1/x
 * with x = u.  Lets a test compare the device forms (hardware seeds) with libm directly. */
int qcd_debug_hb_math(const uint32_t* words, size_t n, double* out);

/* Profiling (QCD_OPT_PROFILE = 1): summed device time (ms, CUDA events on the lattice's stream) and launch count of
 * the update kernels of `kind` since the last qcd_reset_profile.  Synchronises the stream. */
int qcd_get_profile(qcd_lattice_t* lat, int kind, double* total_ms, uint64_t* launches);
int qcd_reset_profile(qcd_lattice_t* lat);
/* Number of kernels this library launched for the lattice since creation . */
int qcd_get_launch_count(qcd_lattice_t* lat, uint64_t* out);

/* Peaks measured on the current device, for the roofline denominators (north_star: "peaks measured in the same
 * run").  fma: register-resident FMA chains, result in TFLOP/s (2 flop per FMA).  copy: device-to-device copy of
 * `bytes` bytes, best of `reps`, result in GB/s counting read + write bytes.  Both synchronise the device. */
int qcd_probe_fma_tflops(int precision, double* tflops);
int qcd_probe_copy_gbs(size_t bytes, int reps, double* gbs);

/* ---------------------------------------------------------------------------------------------------------------------
 * A lattice divided into parts.  PAPER.md:124-128 sec 4: "dividing lattice is made into unequal parts
 * ... in first spatial coordinate direction ... Divided lattice simulation differs from a full lattice simulation only in
 * necessity to carry out the exchanging values of boundary sites"; used for several devices and when one device's memory
 * is not enough.  Here the split direction is the slowest SPATIAL direction, dims[D-2] (D >= 3), so that a part holds whole
 * time lines (the Polyakov loop stays local).  A part ("slab") of `extent` layers starting at global coordinate `offset`
 * (both even) is a qcd_lattice_t of local extent extent + 2 along that direction: its own layers, then a copy of the next
 * part's first layer and a copy of the previous part's last layer (one-site link halos: a staple reaches one site).
 * After every (parity, mu) sub-step the two boundary layers of the array that sub-step wrote are copied to the neighbours
 * (qcd_split_*: by the update kernel itself, which stores a boundary link a second time into the neighbouring part's
 * memory -- a peer GPU's with one part per device; slab primitives: by qcd_slab_halo_pack / unpack).
 * The Philox counters use the GLOBAL site index, so a divided lattice reproduces the undivided one bit for bit.
 * A part's halo copies are written by its NEIGHBOURS' kernels on their streams: they are valid on the part's own stream only
 * behind a wait for the neighbours' last update (qcd_split_substep, qcd_split_sweep and qcd_split_measure enqueue that wait
 * themselves; qcd_split_destroy drains every part's stream before it frees anything).
 *
 * Slab primitives (one part per handle; the parts may live in different processes, one per GPU, and exchange the packed
 * layers through any transport, e.g. torch.distributed / NCCL):
 *   qcd_slab_bytes / qcd_slab_create   like qcd_lattice_bytes / qcd_lattice_create, dims = GLOBAL extents.
 *   qcd_init, qcd_set_links / qcd_get_links (canonical layout of the part's own block, lex order of its own extents),
 *   qcd_debug_substep (updates the part's own sites), qcd_set/get_seed, qcd_set/get_sweep_counter work on a slab;
 *   qcd_sweep, qcd_sweep_measure, qcd_measure, qcd_measure_accumulate return QCD_ERR_UNSUPPORTED on it.
 *   qcd_slab_halo_bytes                bytes of one boundary layer of one (parity, mu) array.
 *   qcd_slab_halo_pack(side)           side 0: the first own layer, side 1: the last own layer -> DEVICE buffer.
 *   qcd_slab_halo_unpack(side)         DEVICE buffer -> side 0: the copy of the previous part's last layer,
 *                                      side 1: the copy of the next part's first layer.  Both asynchronous on the stream.
 *   qcd_slab_measure_sums              SUMS over the part's own sites of (1/N) Re Tr plaquette per plane and of
 *                                      (1/N) Tr Polyakov line (either may be NULL); synchronises.  The caller adds the
 *                                      parts and divides by V resp. V / dims[D-1].
 * Split driver (all parts in this process; devices[k] = CUDA device of part k, NULL = the current device for all; parts on
 * different devices need peer access and write each other's halo layers directly over NVLink):
 *   qcd_split_create(extents = NULL: parts as equal as even extents allow), qcd_split_init, qcd_split_sweep,
 *   qcd_split_substep, qcd_split_measure, qcd_split_get_links / qcd_split_set_links (HOST, global canonical layout),
 *   qcd_split_set_seed, qcd_split_set/get_sweep_counter, qcd_split_parts, qcd_split_halo_bytes (bytes copied between
 *   parts per sub-step), qcd_split_synchronize, qcd_split_destroy.  Same argument rules and errors as the undivided calls.
 * ------------------------------------------------------------------------------------------------------------------- */
typedef struct qcd_split qcd_split_t;
size_t qcd_slab_bytes(int D, const int* dims, int Nc, int precision, unsigned flags, int offset, int extent);
int qcd_slab_create(int D, const int* dims, int Nc, int precision, unsigned flags, int offset, int extent, void* device_mem,
                    size_t bytes, void* cuda_stream, qcd_lattice_t** out);
size_t qcd_slab_halo_bytes(qcd_lattice_t* lat);
int qcd_slab_halo_pack(qcd_lattice_t* lat, int parity, int mu, int side, void* device_buf, size_t bytes);
int qcd_slab_halo_unpack(qcd_lattice_t* lat, int parity, int mu, int side, const void* device_buf, size_t bytes);
int qcd_slab_measure_sums(qcd_lattice_t* lat, const qcd_field_t* field, double* plaq_sums, double* polyakov_sum);
int qcd_split_create(int D, const int* dims, int Nc, int precision, unsigned flags, int n_parts, const int* extents,
                     const int* devices, qcd_split_t** out);
int qcd_split_destroy(qcd_split_t* s);
int qcd_split_parts(qcd_split_t* s, int* n_parts, int* offsets, int* extents, int capacity);
int qcd_split_halo_bytes(qcd_split_t* s, size_t* per_substep);
int qcd_split_init(qcd_split_t* s, int start, uint64_t seed);
int qcd_split_sweep(qcd_split_t* s, double beta, int n_hb, int n_or, const qcd_field_t* field);
int qcd_split_substep(qcd_split_t* s, double beta, int kind, int hit, int parity, int mu, const qcd_field_t* field);
int qcd_split_measure(qcd_split_t* s, const qcd_field_t* field, double* plaq_total, double* plaq_planes, double* polyakov_re_im);
int qcd_split_get_links(qcd_split_t* s, void* dst, size_t bytes);
int qcd_split_set_links(qcd_split_t* s, const void* src, size_t bytes);
int qcd_split_set_seed(qcd_split_t* s, uint64_t seed);
int qcd_split_set_sweep_counter(qcd_split_t* s, uint32_t value);
int qcd_split_get_sweep_counter(qcd_split_t* s, uint32_t* out);
int qcd_split_synchronize(qcd_split_t* s);

/* ---------------------------------------------------------------------------------------------------------------------
 * The O(N) scalar model on lattice sites, the paper's second workload: "In case of O(N)
 * models the fields are set with N-vectors, which are associated with lattice sites", :108 "Improved Metropolis algorithm
 * [7] is used for O(N) update", :134 "For O(4) model NHIT=100 tries were used to update each lattice site".  Ref [7] (the
 * N-component lambda phi^4 model) is not available; readings R16-R19 of DESIGN.md:
 *   action  S = sum_x [ -2 kappa sum_mu phi(x).phi(x+mu) + phi(x).phi(x) + lambda (phi(x).phi(x) - 1)^2 ]
 *   sweep   for parity in (0, 1): every site of that parity makes nhit Metropolis tries phi' = phi + delta (2u - 1) per
 *           component, accepted iff u' < exp(-(S(phi') - S(phi))), each from its current value, all nhit made; then the sweep
 *           counter is incremented.  One Philox4x32-10 block per try, counter (lex site, sweep counter,
 *           parity<<4 | try<<8 | 2<<24, 0): five 23-bit numbers, u = (k + 1/2) 2^-23.  N = 1..4, D = 2..4, extents even.
 *   starts  QCD_COLD: phi = (1, 0, .., 0); QCD_HOT: components uniform in (-1, 1) from Philox domain 3.
 * Canonical field layout (get/set): [lex site][component] in the lattice's precision.  Handles, memory, streams, status codes
 * and asynchrony as for qcd_lattice_t; qcd_on_measure, qcd_on_get_counts and host transfers synchronise the stream.
 * qcd_on_measure: phi2 = (1/V) sum phi.phi, link = (1/(V D)) sum_x sum_mu phi(x).phi(x+mu), mag[N] = (1/V) sum phi (any may be
 * NULL).  qcd_on_get_counts: accepted and made tries since qcd_on_init.  qcd_on_half_sweep: one parity, counter unchanged.
 * ------------------------------------------------------------------------------------------------------------------- */
typedef struct qcd_on qcd_on_t;
size_t qcd_on_bytes(int D, const int* dims, int N, int precision);
int qcd_on_create(int D, const int* dims, int N, int precision, void* device_mem, size_t bytes, void* cuda_stream, qcd_on_t** out);
int qcd_on_destroy(qcd_on_t* lat);
int qcd_on_init(qcd_on_t* lat, int start, uint64_t seed);
int qcd_on_sweep(qcd_on_t* lat, double kappa, double lambda, double delta, int nhit);
int qcd_on_half_sweep(qcd_on_t* lat, int parity, double kappa, double lambda, double delta, int nhit);
int qcd_on_measure(qcd_on_t* lat, double* phi2, double* link, double* mag);
int qcd_on_get_counts(qcd_on_t* lat, uint64_t* accepted, uint64_t* tried);
int qcd_on_get_field(qcd_on_t* lat, void* dst, size_t bytes, int dst_is_device);
int qcd_on_set_field(qcd_on_t* lat, const void* src, size_t bytes, int src_is_device);
int qcd_on_set_seed(qcd_on_t* lat, uint64_t seed);
int qcd_on_set_sweep_counter(qcd_on_t* lat, uint32_t value);
int qcd_on_get_sweep_counter(qcd_on_t* lat, uint32_t* out);

const char* qcd_last_error(void);
const char* qcd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* QCD_B200_H */
