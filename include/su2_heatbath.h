/*
 * su2_heatbath.h — C ABI of the B200 (sm_100a) SU(2) pure-gauge heat-bath library.
 *
 * The library implements the data-parallel hot path of arxiv/paper_1104_5432
 * ("Finite temperature lattice QCD with GPUs"): random SU(2) initialisation,
 * checkerboarded heat-bath sweeps, the mean plaquette (§2.1) and the
 * Polyakov loop (eq. 1). The paper prints no formula for the
 * update; the readings [R1]..[R14] that define it are in DESIGN.md §3 (they restate
 * SURVEY.md §8(c) and BASELINE.json north_star).
 *
 * General conventions
 *  - Every call returns an int status: SU2_OK or one of the SU2_E* codes below.
 *    No exception crosses the ABI, nothing calls exit().
 *  - `su2_lattice*` is an opaque handle owned by the caller from create to destroy.
 *    A handle is not thread-safe; different handles are independent. No global state.
 *  - DEVICE pointers are marked [device], HOST pointers [host]. Out-pointers are
 *    caller-owned.
 *  - Lattice N_x x N_y x N_z x N_t, periodic, V sites; directions mu = 0,1,2,3 = x,y,z,t.
 *    Site index s = x + N_x (y + N_y (z + N_z t)); parity p = (x+y+z+t) & 1.
 *  - A link is a unit quaternion a = (a0,a1,a2,a3), U = a0 + i(a1 s1 + a2 s2 + a3 s3) [R1].
 *  - Canonical HOST order of a configuration: [t][z][y][x][mu][4], i.e. element
 *    ((s*4 + mu)*4 + c), real type = the lattice precision (float or double).
 *  - DEVICE layout: 8 arrays indexed [p][mu], each V/2 quaternions,
 *    element index h = s >> 1; array (p,mu) starts at quaternion (p*4+mu)*V/2.
 *  - Work is enqueued on the handle's CUDA stream. Calls that return a value to the
 *    host synchronise that stream; su2_heatbath_sweep and su2_init are asynchronous.
 */
#ifndef SU2_HEATBATH_H
#define SU2_HEATBATH_H

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define SU2_API __attribute__((visibility("default")))
#else
#define SU2_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

#define SU2_OK 0      /* success */
#define SU2_EARG 1    /* bad argument (odd/too-small extent, bad precision/start, beta<=0 or
                         non-finite, NULL pointer, wrong byte count) */
#define SU2_EALLOC 2  /* device allocation failed */
#define SU2_ECUDA 3   /* CUDA runtime error; sticky, message via su2_last_error */
#define SU2_ESTATE 4  /* sweep or measurement before su2_init / su2_set_links */
#define SU2_ETOOBIG 5 /* su2_mean_plaquette_noalloc only: lattice larger than its static scratch serves */

#define SU2_START_COLD 0
#define SU2_START_HOT 1

typedef struct su2_lattice su2_lattice;

/* Bytes of device memory one configuration needs: 4*V quaternions of the precision.
 * Returns 0 for invalid arguments. */
SU2_API size_t su2_lattice_bytes(int Nx, int Ny, int Nz, int Nt, int precision);

/* Create a lattice on the current CUDA device; the library allocates (cudaMalloc) the
 * links and its reduction scratch and creates nothing else; work runs on the legacy
 * default stream unless su2_set_stream is called.
 *   precision: 32 (float4 links) or 64 (double links).
 *   Each extent must be even and >= 2 (checkerboard + periodic wrap [R4]); V < 2^32
 *   (the site index is one 32-bit Philox counter word [R5]).
 * *out receives the handle. Errors: SU2_EARG, SU2_EALLOC, SU2_ECUDA. */
SU2_API int su2_lattice_create(int Nx, int Ny, int Nz, int Nt, int precision, su2_lattice** out);

/* As above, but the caller owns the link storage ("PyTorch owns memory"):
 *   dev_links  [device] buffer of `bytes` >= su2_lattice_bytes(...), 32-byte aligned;
 *              the library never frees it and it must outlive the handle.
 *   cuda_stream a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream), may be 0.
 * The small reduction scratch is still allocated by the library. */
SU2_API int su2_lattice_create_external(int Nx, int Ny, int Nz, int Nt, int precision, void* dev_links,
                                size_t bytes, void* cuda_stream, su2_lattice** out);

/* Free what the library allocated. NULL is a no-op (returns SU2_OK). */
SU2_API int su2_lattice_destroy(su2_lattice* lat);

/* Change the stream later work is enqueued on (cudaStream_t, may be 0). */
SU2_API int su2_set_stream(su2_lattice* lat, void* cuda_stream);

/* Row 1 of the path ("random SU(2) matrix initialization") [R9].
 *   start = SU2_START_COLD: every link = (1,0,0,0).
 *   start = SU2_START_HOT : Haar-random unit quaternion per link from
 *           Philox4x32-10(counter = (s, 0, (1<<8)|(p<<2)|mu, 0), key = seed).
 * Stores `seed` in the handle; it keys every later draw. Asynchronous. */
SU2_API int su2_init(su2_lattice* lat, int start, uint64_t seed);

/* Set the seed that keys later sweeps without touching the links (resume from a
 * configuration loaded with su2_set_links). Takes effect for every later call, su2_run included. */
SU2_API int su2_set_seed(su2_lattice* lat, uint64_t seed);

/* Launch-structure switches of a handle. They change HOW the kernels are
 * launched, never what they compute: results are bit-identical with either value (GPU tests).
 *   SU2_OPT_OVERLAP   1 (default): consecutive sub-steps of a sweep are chained by programmatic
 *                     dependent launch; 0: every launch fully serialised behind its predecessor.
 *   SU2_OPT_RUN_GRAPH 1 (default): su2_run replays one captured CUDA graph per step; 0: it enqueues
 *                     the step's kernels directly.
 *   SU2_OPT_TAIL_OVERLAP (default: automatic - on for lattices of a few CTA waves per sub-step, i.e. below ~5 M sites,
 *                     off above; 0 / 1 force it): inside su2_run the Polyakov kernel of step i (which also finishes the
 *                     step's two observables) runs on a second private stream beside the first six sub-steps
 *                     of step i+1 - it reads only U_t, which step i+1 writes from its seventh sub-step on - and
 *                     is joined before that sub-step; the fused-plaquette partials and the device loop state
 *                     alternate between two sets, and a captured graph holds 16 steps. Worth 5-23 % of a
 *                     step from 8^4 to 32^4, neutral at 48^3 x 8 .. 48^4, costs 4 % at 64^4.
 *                     dev_out is complete when su2_run's work on the handle's stream is (as without the option).
 * value must be 0 or 1. Errors: SU2_EARG. */
#define SU2_OPT_OVERLAP 0
#define SU2_OPT_RUN_GRAPH 1
#define SU2_OPT_TAIL_OVERLAP 2
SU2_API int su2_set_option(su2_lattice* lat, int option, int value);

/* Rows 2-6: one full heat-bath sweep = the 8 sub-steps (mu = 0..3 outer, parity 0,1
 * inner) [R4]; each sub-step updates every U_mu(x) of that parity from its Wilson
 * staple sum [R3] with a Kennedy-Pendleton draw [R6][R7], random numbers from
 * Philox4x32-10(counter = (s, sweep_idx, (p<<2)|mu, n), key = seed) [R5].
 * Same (links, seed, beta, sweep_idx) => same result on any launch geometry.
 * The caller must not reuse a sweep_idx within a run. Asynchronous.
 * Errors: SU2_EARG (beta <= 0 or not finite), SU2_ESTATE, SU2_ECUDA. */
SU2_API int su2_heatbath_sweep(su2_lattice* lat, double beta, uint32_t sweep_idx);

/* S8(f) NEXT-3(i), north_star "Creutz/Kennedy-Pendleton" [R15]: which draw of x0 (density
 * ~ sqrt(1-x0^2) exp(alpha x0), alpha = beta k) later sweeps of this handle use.
 *   SU2_DRAW_KP     Kennedy-Pendleton on every link [R6] (the default; alpha >= 5 on every
 *                   BASELINE config, acceptance 0.93-0.99)
 *   SU2_DRAW_CREUTZ Creutz's original draw on every link: trial n = 1,2,...: (R, R', ., .) =
 *                   u(words of Philox(..., n)); delta = -ln(R + (1-R) exp(-2 alpha))/alpha;
 *                   accept iff R'^2 <= delta (2 - delta); x0 = 1 - delta. Acceptance
 *                   (pi/2) I1(alpha)/sinh(alpha): 0.76 at alpha = 1, 0.22 at alpha = 32.
 *   SU2_DRAW_AUTO   per link: Creutz iff alpha < SU2_ALPHA_C (where the two acceptances
 *                   are equal), else KP. For strong coupling (beta <~ 0.5).
 * Direction, composition [R7] and the Philox keying [R5] are the same for both.
 * Errors: SU2_EARG. */
#define SU2_DRAW_KP 0
#define SU2_DRAW_AUTO 1
#define SU2_DRAW_CREUTZ 2
#define SU2_ALPHA_C 1.6847
SU2_API int su2_set_draw(su2_lattice* lat, int method);

/* One sub-step (mu, parity) only — the unit the tests compare against the oracle. */
SU2_API int su2_heatbath_substep(su2_lattice* lat, double beta, uint32_t sweep_idx, int mu, int parity);

/* Row 7: P = 1/(6V) sum_x sum_{mu<nu} 1/2 Tr U_mu(x) U_nu(x+mu) U_mu^dag(x+nu)
 * U_nu^dag(x) [R10]; fp64 accumulation in a fixed order. Synchronises; *out [host] in [-1,1]. */
SU2_API int su2_mean_plaquette(su2_lattice* lat, double* out);

/* Row 8 (eq. 1): signed spatial average of
 * 1/2 Tr prod_{t=0}^{N_t-1} U_t(x,t) [R11]. Synchronises; *out [host]. */
SU2_API int su2_polyakov_loop(su2_lattice* lat, double* out);

/* Rows 7+8 with one synchronisation: enqueue both reductions, then copy both doubles.
 * Either out pointer may be NULL to skip that measurement. */
SU2_API int su2_measure(su2_lattice* lat, double* plaquette_out, double* polyakov_out);

/* Asynchronous form used for per-sweep measurement without a host round trip:
 * enqueue the plaquette (slot 0) and Polyakov (slot 1) reductions of the current
 * configuration and store the two doubles at dev_out[2*index], dev_out[2*index+1]
 * ([device], caller-owned). No synchronisation. */
SU2_API int su2_measure_async(su2_lattice* lat, double* dev_out, size_t index);

/* The paper's loop body in one call ("100 iterations of the heat bath method and
 * the calculation of the mean average plaquette at each iteration"): one sweep exactly as
 * su2_heatbath_sweep, then the mean plaquette [R10] and the Polyakov loop [R11] of the NEW
 * configuration at dev_out[2*index], dev_out[2*index+1] ([device], caller-owned doubles).
 * The plaquette is accumulated inside the sub-steps (mu >= 1, parity 1) as 1/2 Tr(U' w), w =
 * the staple terms of the directions nu < mu, which sums every plaquette of the final
 * configuration once; it equals su2_mean_plaquette after the sweep to rounding
 * (fp64 accumulation, fixed order) and saves that kernel's pass over the lattice.
 * event_after_sweep: NULL, or a cudaEvent_t the library records on the handle's stream
 * between the 8th sub-step and the two reduction kernels (bench.py times the sub-steps with it).
 * Asynchronous, no synchronisation. Errors as su2_heatbath_sweep, plus SU2_EARG for NULL dev_out. */
SU2_API int su2_heatbath_sweep_measure(su2_lattice* lat, double beta, uint32_t sweep_idx, double* dev_out,
                                       size_t index, void* event_after_sweep);

/* The paper's whole loop in one call (N iterations of heat bath + plaquette):
 * n_steps times { su2_heatbath_sweep_measure(beta, sweep_idx0 + i) } with the results of step i
 * at dev_out[2*i] (mean plaquette) and dev_out[2*i+1] (Polyakov loop); dev_out [device] holds
 * 2*n_steps doubles. One step is captured once per handle as a CUDA graph (10 kernels, the
 * sub-steps chained by programmatic dependent launch) and replayed; sweep index, 1/beta and the
 * output slot live in device memory, so no kernel parameter changes between replays
 * (DESIGN.md 6.6). Same links and observables as the step-by-step calls, bit for bit.
 * Runs on a private stream ordered after, and joined back into, the handle's stream.
 * Asynchronous. Errors: SU2_EARG (beta, NULL dev_out), SU2_ESTATE, SU2_ECUDA. */
SU2_API int su2_run(su2_lattice* lat, double beta, uint32_t sweep_idx0, uint32_t n_steps, double* dev_out);

/* S8(f) NEXT-2: replica batches. The paper's production mode is many small finite-temperature
 * lattices, one per coupling (a beta scan per N_t); a 16^3 x 4 sub-step is 64 CTAs on a
 * 148-SM GPU. A batch handle holds n_replicas configurations of the same geometry and precision, one
 * after the other in device memory (replica r at byte offset r * su2_lattice_bytes(...)), and
 * su2_batch_sweep_measure updates all of them with the same 9 launches a single lattice takes, each
 * replica with its own beta and its own seed (its Philox streams are those of a single lattice with that
 * seed).
 *   1 <= n_replicas <= 65535; n_replicas * 4V < 2^32 (every link of the batch has a 32-bit index).
 * Every single-lattice call (init, sweep, measure, correlator, get/set_links, run ...) works on a batch
 * handle and acts on the SELECTED replica (0 after create). The _external form takes caller-owned
 * memory of n_replicas * su2_lattice_bytes(...) bytes. */
SU2_API int su2_lattice_create_batch(int Nx, int Ny, int Nz, int Nt, int precision, int n_replicas,
                                     su2_lattice** out);
SU2_API int su2_lattice_create_batch_external(int Nx, int Ny, int Nz, int Nt, int precision, int n_replicas,
                                              void* dev_links, size_t bytes, void* cuda_stream, su2_lattice** out);
/* Number of replicas of the handle (1 for su2_lattice_create); 0 for NULL. */
SU2_API int su2_replicas(const su2_lattice* lat);
/* Make replica `replica` the one the single-lattice calls act on. Errors: SU2_EARG. */
SU2_API int su2_select_replica(su2_lattice* lat, int replica);
/* su2_init of every replica: replica r from seeds[r] ([host], n_replicas values). Asynchronous. */
SU2_API int su2_batch_init(su2_lattice* lat, int start, const uint64_t* seeds);
/* One step (heat-bath sweep [R4], mean plaquette [R10], Polyakov loop [R11]) of every replica:
 * replica r at coupling betas[r] ([host], n_replicas values), Philox counter word sweep_idx for all.
 * Results at dev_out[2*(index*n_replicas + r)], dev_out[2*(index*n_replicas + r) + 1] ([device]).
 * The draw is the handle's (su2_set_draw). Asynchronous, except that a change of betas or seeds since
 * the previous call first waits for the stream. Errors: SU2_EARG, SU2_ESTATE (a replica not
 * initialised), SU2_ECUDA. */
SU2_API int su2_batch_sweep_measure(su2_lattice* lat, const double* betas, uint32_t sweep_idx, double* dev_out,
                                    size_t index);
/* su2_run for a batch: n_steps rounds of su2_batch_sweep_measure(betas, sweep_idx0 + i, dev_out, i) as one call - the
 * beta scan of PAPER.md:63-72 as the paper's loop. One round (9 launches) is captured once per handle as a
 * CUDA graph and replayed; the sweep index and the output slot live in device memory, couplings and seeds in the
 * per-replica device table. dev_out [device] holds 2 * n_replicas * n_steps doubles: step i of replica r at
 * dev_out[2*(i*n_replicas + r)] (plaquette) and + 1 (Polyakov loop). Same links and observables as the round-by-round
 * calls, bit for bit. Runs on the private stream of su2_run, ordered after and joined back into the handle's stream.
 * Asynchronous (a change of betas or seeds first waits for the stream). Errors as su2_batch_sweep_measure. */
SU2_API int su2_batch_run(su2_lattice* lat, const double* betas, uint32_t sweep_idx0, uint32_t n_steps, double* dev_out);

/* NEXT-1 (eq. 3): on-axis Polyakov-loop correlator
 * C(r) = < l(x) l(x + r e_i) >, averaged over all spatial x and the 3 spatial axes i,
 * r = 1..rmax (rmax <= min spatial extent / 2), l(x) = 1/2 Tr L(x) (real in SU(2)).
 * out [host] receives rmax doubles. Synchronises. */
SU2_API int su2_polyakov_correlator(su2_lattice* lat, int rmax, double* out);

/* Configuration I/O in canonical host order (see top). bytes must equal
 * su2_lattice_bytes(...). Both synchronise. su2_set_links marks the lattice initialised.
 * host pointers may be pageable or pinned. su2_get_links, like su2_synchronize and the measuring
 * calls, returns SU2_ECUDA if a kernel of the run raised a device-side flag (Kennedy-Pendleton
 * trial cap; in a -DHB_BOUNDS_CHECK build, a link index outside its array): host_dst is then
 * filled all the same, the message says which flag. */
SU2_API int su2_get_links(su2_lattice* lat, void* host_dst, size_t bytes);
SU2_API int su2_set_links(su2_lattice* lat, const void* host_src, size_t bytes);

/* Block until all work enqueued on the handle's stream has finished. */
SU2_API int su2_synchronize(su2_lattice* lat);

/* ---------------------------------------------------------------------------------------
 * S8(f) NEXT-4: the lattice split into time slabs, one per GPU — the paper's second mode
 * ("2 GPUs ... OpenMP"; the exchange itself is not described there;
 * SURVEY.md §8(e) states it; DESIGN.md §6.9 is the design). Not part of the benchmarked path.
 *
 * A slab owns the Lt global time slices t0 .. t0+Lt-1 (t0, Lt even, Lt >= 2) of an
 * Nx x Ny x Nz x Nt lattice and stores Lt + 4 local slices: local slice t is a copy of global
 * slice (t0 - 2 + t) mod Nt; slices 2 .. Lt+1 are the interior (updated here), slices 1 and Lt+2
 * are the halos the staples read (owned by the slab below / above), slices 0 and Lt+3 are
 * padding that keeps local and global site parity equal. The handle is an ordinary lattice of
 * local extents Nx x Ny x Nz x (Lt+4) as far as memory goes: same device layout with V = local
 * sites, and su2_get_links / su2_set_links move the Lt+4 local slices in canonical order.
 *
 * One sub-step (mu, parity) of the whole lattice = su2_slab_substep on every slab, in any order or
 * concurrently, then a barrier: the kernel that updates a slab's first / last interior slice also
 * stores those links into the halo of the slab below / above (plain stores into peer memory over
 * NVLink, or into another buffer of the same device), so there is no separate exchange step, and
 * within a sub-step no slab reads what another one writes. Draws are keyed by the GLOBAL site [R5]:
 * the result is the one su2_heatbath_substep gives on the unsplit lattice, bit for bit.
 * The whole-lattice calls (su2_heatbath_sweep, su2_heatbath_sweep_measure, su2_run, su2_measure*,
 * su2_polyakov_correlator, su2_batch_*) return SU2_ESTATE on a slab handle; su2_init (every local
 * slice, halos included, from its global site), su2_set_seed, su2_set_draw, su2_set_stream,
 * su2_heatbath_substep (= su2_slab_substep without the fused plaquette), su2_get/set_links work. */
SU2_API size_t su2_slab_bytes(int Nx, int Ny, int Nz, int Lt, int precision); /* 0 = invalid */
SU2_API int su2_slab_create(int Nx, int Ny, int Nz, int Nt, int precision, int t0, int Lt, su2_lattice** out);
SU2_API int su2_slab_create_external(int Nx, int Ny, int Nz, int Nt, int precision, int t0, int Lt, void* dev_links,
                                     size_t bytes, void* cuda_stream, su2_lattice** out);

/* Where the edge slices are also stored: lo_links / hi_links [device, this or a peer device] = the
 * link buffers (su2_device_links) of the slabs that own global slices t0-1 and t0+Lt (periodic; with
 * two slabs both are the other slab, with one slab both are the handle's own buffer), lo_Lt / hi_Lt
 * their interior extents. The buffers must stay valid while sub-steps run. Errors: SU2_EARG, SU2_ESTATE. */
SU2_API int su2_slab_set_peers(su2_lattice* lat, void* lo_links, int lo_Lt, void* hi_links, int hi_Lt);

/* Rows 2-6 on the interior slices + the stores into the neighbours' halos. fuse_plaquette != 0: the
 * sub-steps (mu >= 1, parity 1) also keep the plaquette partials of their planes.
 * Asynchronous. The caller provides the barrier between sub-steps (stream order on one device; a
 * stream-ordered collective or an event across devices). */
SU2_API int su2_slab_substep(su2_lattice* lat, double beta, uint32_t sweep_idx, int mu, int parity, int fuse_plaquette);

/* Row 7 on a slab: *dev_out [device] = (sum over the plaquettes based at interior sites) / (6 V_global),
 * so the values of all slabs add up to the mean plaquette [R10]. fused != 0: from the partials of
 * the last sweep's fused sub-steps; else by the plaquette kernel (needs a current upper halo).
 * Asynchronous. */
SU2_API int su2_slab_plaquette(su2_lattice* lat, int fused, double* dev_out);

/* Row 8 across slabs [R11]: the ordered product of the time links continues from slab to slab.
 *   dev_prev [device] NxNyNz links (the product over all slices below t0, per spatial site, index
 *            x + Nx (y + Ny z)), NULL exactly on the slab with t0 = 0;
 *   dev_next [device, nullable] receives the product including this slab's slices;
 *   dev_out  [device, nullable] receives the spatial mean of 1/2 Tr of that product (the Polyakov
 *            loop when this is the last slab).
 * Same left-to-right association as the single-lattice loop. Asynchronous. */
SU2_API int su2_slab_polyakov(su2_lattice* lat, const void* dev_prev, void* dev_next, double* dev_out);

/* CUDA IPC plumbing for one process per GPU: export the (library-allocated: su2_slab_create) link
 * buffer as a 64-byte handle [host]; open / close such a handle in another process. su2_ipc_open
 * returns a [device] pointer valid in the calling process for su2_slab_set_peers. */
SU2_API int su2_ipc_export(su2_lattice* lat, void* handle64);
SU2_API int su2_ipc_open(const void* handle64, void** dev_ptr);
SU2_API int su2_ipc_close(void* dev_ptr);

/* Row 7 ([R10]) WITHOUT ANY ALLOCATION: for callers that cannot call cudaMalloc - code under CUDA graph
 * capture, tight serving loops, harnesses that forbid it. No handle (creating one allocates): the caller passes the
 * configuration and the destination, the call enqueues the plaquette kernel and a final sum on cuda_stream (a
 * cudaStream_t, may be 0) and calls no cudaMalloc, cudaFree or allocating library routine.
 *   dev_links [device] a configuration in DEVICE layout (see top: 8 arrays [p][mu] of V/2 quaternions of the
 *             precision; what su2_device_links returns / what a caller-owned buffer of a handle holds), 32-byte aligned;
 *   dev_out   [device] receives the mean plaquette (one double) when the stream reaches it. Asynchronous.
 * The per-CTA partial sums - library-allocated per handle everywhere else - live in ONE file-scope static device
 * array of 2^18 doubles (2 MiB, held by every GPU that loads the library until exit), which serves lattices of up to
 * SU2_NOALLOC_MAX_SITES = 2^25 sites (64^4 = 2^24). All calls share it: calls that can overlap on the GPU (different
 * streams, no ordering between them) race and give wrong results; calls on one stream, or otherwise ordered, are safe.
 * Nothing in it has to start at zero (each call writes every partial it reads), so it is never cleared.
 * Same kernels, same fixed reduction order as su2_mean_plaquette: the same bits for the same configuration.
 * Errors: SU2_EARG (NULL or misaligned pointer, bad extents or precision), SU2_ETOOBIG (V > SU2_NOALLOC_MAX_SITES;
 * nothing is launched), SU2_ECUDA (launch failure). */
#define SU2_NOALLOC_MAX_SITES (1u << 25)
SU2_API int su2_mean_plaquette_noalloc(const void* dev_links, int Nx, int Ny, int Nz, int Nt, int precision,
                                       void* cuda_stream, double* dev_out);

/* Measurement support: memory bandwidth of the current device with the
 * access shape of the path - 128-bit loads, unit stride across a warp, every SM busy, no arithmetic - over a
 * zero-filled scratch buffer of `bytes` (>= 1 MiB, multiple of 32) that the call allocates and frees.
 *   mode SU2_PROBE_READ: every pass reads the buffer once. With bytes <= L2 (64 MiB = the 32^4 fp32 lattice
 *        in the 126 MB L2) the passes after the two untimed ones are served by L2: the L2 roofline
 *        denominator of the cache-resident point of the metric. With bytes >> L2: HBM read bandwidth.
 *   mode SU2_PROBE_COPY: every pass copies the first half onto the second (read + write = `bytes`).
 * *gbs_out [host] = bytes per pass / mean duration of `passes` passes (CUDA events on cuda_stream, may
 * be 0), in GB/s (1e9); *us_per_pass_out [host, nullable]. Synchronises that stream.
 * Errors: SU2_EARG, SU2_EALLOC, SU2_ECUDA. No handle: nothing of a lattice is touched. */
#define SU2_PROBE_READ 0
#define SU2_PROBE_COPY 1
SU2_API int su2_bandwidth_probe(size_t bytes, int passes, int mode, void* cuda_stream, double* gbs_out,
                                double* us_per_pass_out);

/* Number of kernels this handle has launched so far (bench.py's gpu_launches). */
SU2_API uint64_t su2_launch_count(const su2_lattice* lat);

/* [device] pointer to the links in device layout (for callers that own the memory
 * model; NULL on a NULL handle). */
SU2_API void* su2_device_links(su2_lattice* lat);

/* Message of the last error on this handle ("" if none); static string for a code. */
SU2_API const char* su2_last_error(const su2_lattice* lat);
SU2_API const char* su2_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* SU2_HEATBATH_H */
