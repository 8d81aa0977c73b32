/* gcoreccd.h — C ABI of the B200-native (sm_100a) hot path of G-CoReCCD (arXiv 2203.11043).
 *
 * One handle = one event (one set of mutually interacting holes) = one CUDA stream; or, through the
 * *_events calls, one batch of independent small events advanced concurrently.
 * Per time step the library runs, entirely on the GPU and in this order (Fig. 2):
 *   a1  all-pairs softened Coulomb field of every still-drifting hole      (eq. 6)
 *   a2  + linear depletion field E(z) = a1 z - a2, total |E|               (eq. 1)
 *   a3  hole mobility mu(|E|, T)                                           (eq. 2)
 *   a4  drift  dr = mu E dt
 *   a5  isotropic Gaussian diffusion, sigma^2 = 2 D_h dt, D_h = k_B mu T/q (eqs. 3-4),
 *       normals from Philox4x32-10 keyed by (seed, carrier id, step)
 *   a6  position update, specular reflection at the back surface
 *   a7  collection test z <= z_well and integer pixel histogram
 *   a8  stable compaction of the carriers still drifting
 *
 * Units: length um, time ns, field V/cm, temperature K.  Positions are FP32 ("3N floats").
 *
 * Conventions
 *   - every function returns 0 (GCORECCD_OK) or a negative gcoreccd_status; run_to_collection may return
 *     +1 (GCORECCD_MAX_STEPS) when max_steps was reached with carriers left ("maximum number
 *     of iterations"), which is not an error.
 *   - pointers named *_host are host pointers; pointers with an `on_device` flag are host pointers when
 *     the flag is 0 and device pointers (on the handle's device) when it is 1.  All output buffers are
 *     caller-allocated; the library copies inputs and never keeps a caller pointer, except `workspace`.
 *   - no exceptions, no printing, no global state.  A handle is not thread-safe; distinct handles are
 *     independent.  There is NO CPU fallback: create() fails with GCORECCD_ERR_CUDA without an sm_100 GPU.
 *   - gcoreccd_step is asynchronous on the handle's stream; every function that returns data to the host
 *     synchronises that stream first.
 */
#ifndef GCORECCD_H
#define GCORECCD_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct gcoreccd gcoreccd_t;

typedef enum {
  GCORECCD_OK            = 0,
  GCORECCD_MAX_STEPS     = 1,
  GCORECCD_ERR_INVALID   = -1,   /* bad argument / parameter                         */
  GCORECCD_ERR_STATE     = -2,   /* call not valid in the handle's current state     */
  GCORECCD_ERR_CAPACITY  = -3,   /* more carriers than max_carriers / buffer too small */
  GCORECCD_ERR_NOMEM     = -4,
  GCORECCD_ERR_CUDA      = -5,   /* CUDA runtime error or no sm_100 device           */
  GCORECCD_ERR_NONFINITE = -6    /* a carrier position became NaN/Inf                */
} gcoreccd_status;

enum {                            /* gcoreccd_params.flags */
  GCORECCD_COULOMB_OFF   = 1u,    /* PAPER.md:88 "whether Coulomb repulsion should be computed" */
  GCORECCD_DIFFUSION_OFF = 2u,    /* test hook: deterministic drift                  */
  GCORECCD_DEPLETION_OFF = 4u     /* test hook: a1 = a2 = 0                          */
};

/* Largest capacity of one handle: 2^24 holes (32 B of state + 192 B of partial-sum planes + 16 B of collection record per
 * hole of capacity: 4.0 GB at 2^24).  Tested up to 4,194,304 holes (tests/test_gpu_full_runs.py); one all-pairs step at 2^24
 * holes is 2.8e14 interactions (~100 s on a B200), beyond which the far-field variant or target sharding is the tool. */
#define GCORECCD_MAX_CARRIERS (1ull << 24)

typedef struct {
  uint32_t struct_size;           /* = sizeof(gcoreccd_params); ABI versioning                            */
  uint32_t flags;                 /* bits above; 0 = full physics                                          */
  double   T_K;                   /* > 0, eq. 2 / eq. 4                                                    */
  double   a1_V_per_cm2;          /* eq. 1, z measured from the front surface (z = 0), z in cm             */
  double   a2_V_per_cm;           /* eq. 1                                                                 */
  double   thickness_um;          /* back surface, > z_well_um; carriers are mirrored back at it           */
  double   z_well_um;             /* collection plane ("depth of the potential well")          */
  double   pixel_pitch_um;        /* > 0                                                    */
  double   dt_ns;                 /* > 0                                                                   */
  double   softening_um;          /* eps of eq. 6, >= 0; 0 evaluates eq. 5 (coincident pairs contribute 0) */
  double   eps_si;                /* relative permittivity, 0 => 11.7                                      */
  uint64_t seed;                  /* Philox key                                                            */
  int32_t  img_nx, img_ny;        /* image window in pixels, each in [1, 16384]                            */
  double   img_x0_um, img_y0_um;  /* lower-left corner of pixel (0,0)                                      */
  int32_t  device;                /* CUDA ordinal, -1 = current device                                     */
  int32_t  reserved0;
  void*    stream;                /* cudaStream_t to run on (e.g. torch's current stream); NULL => the
                                     library creates and owns a non-blocking stream                        */
  void*    workspace;             /* optional caller-owned device memory (e.g. a torch uint8 tensor),
                                     256-byte aligned, alive until destroy; NULL => the library allocates */
  uint64_t workspace_bytes;       /* >= gcoreccd_workspace_size(max_carriers, img_nx, img_ny)              */
  uint64_t max_carriers;          /* capacity, 1 .. GCORECCD_MAX_CARRIERS                                  */
} gcoreccd_params;

/* Bytes of device memory a handle needs (state ping-pong, field partials, image, counters). */
uint64_t gcoreccd_workspace_size(uint64_t max_carriers, int32_t img_nx, int32_t img_ny);

/* Create / destroy.  *out is set only on success.  Errors: INVALID (parameter ranges, struct_size),
 * CUDA (no sm_100 device, runtime failure), NOMEM, CAPACITY (workspace too small). */
int gcoreccd_create(const gcoreccd_params* p, gcoreccd_t** out);
int gcoreccd_destroy(gcoreccd_t* h);

/* Drop all carriers, zero image, counters and the step index (parameters are kept). */
int gcoreccd_reset(gcoreccd_t* h);

/* Append n carriers.  xyz_um: interleaved x,y,z FP32, host (on_device=0) or device (=1)
 * pointer; copied.  ids continue in load order.  A carrier with z <= z_well is collected at once;
 * non-finite coordinates or z > thickness => INVALID and nothing is loaded; more than max_carriers in
 * total => CAPACITY.  Synchronises the stream. */
int gcoreccd_load_carriers(gcoreccd_t* h, const float* xyz_um, uint64_t n, int on_device);

/* Restart from an exported snapshot (replaces the active set): positions, ids (must be unique) and the step
 * index the next step will use.  The image and counters are kept; n_loaded becomes max(n_loaded, max id + 1).
 * Validated like load_carriers (INVALID on a non-finite coordinate, z > thickness, or z <= z_well: a snapshot holds
 * ACTIVE carriers only).  On a sharded handle every rank loads the same snapshot.  Host pointers. */
int gcoreccd_load_snapshot(gcoreccd_t* h, const float* xyz_um_host, const uint32_t* id_host, uint64_t n,
                           uint64_t step);

/* Enqueue up to n_steps time steps (a1..a8) on the stream; asynchronous.  A step with no active carrier
 * is a no-op and does not advance the step index. */
int gcoreccd_step(gcoreccd_t* h, uint32_t n_steps);

/* Step until no carrier is drifting or max_steps more steps were taken; synchronous.
 * Returns OK, MAX_STEPS (+1), or NONFINITE/CUDA. */
int gcoreccd_run_to_collection(gcoreccd_t* h, uint64_t max_steps, uint64_t* steps_done, uint64_t* n_active_left);

/* Image, row-major [img_ny][img_nx] counts of collected holes; cap_elems >= nx*ny else CAPACITY.
 * n_out_of_window (host pointer, may be NULL) receives the holes collected outside the window, so that
 * sum(image) + n_out_of_window + n_active == n_loaded always. */
int gcoreccd_read_image(gcoreccd_t* h, uint32_t* out, uint64_t cap_elems, uint64_t* n_out_of_window, int on_device);

/* Introspection (host pointers, any may be NULL).  pair_interactions = sum over executed steps of n_active^2
 * (ordered pairs of eq. 6, self terms included, padding excluded). */
int gcoreccd_get_state(gcoreccd_t* h, uint64_t* step, uint64_t* n_active, uint64_t* n_loaded,
                       uint64_t* n_collected, uint64_t* n_out_of_window, uint64_t* pair_interactions);

/* Active carriers in their current (stable, load-ordered) order: interleaved xyz and ids.  Either output
 * may be NULL.  *n receives the active count; fails with CAPACITY if cap < count.  Same on_device flag for both. */
int gcoreccd_read_carriers(gcoreccd_t* h, float* xyz_um, uint32_t* id, uint64_t cap, uint64_t* n, int on_device);

/* Final positions (the image is "the histogram of the output positions"; "save the final
 * results"): for every carrier id < min(n_loaded, max_carriers), its x,y,z (um) after the step in which it crossed
 * z_well and the index of that step (the current step index for holes collected at load); NaN / 0xFFFFFFFF while it is
 * still drifting.  Host buffers of cap entries (3 floats / 1 uint32 per id), both or neither; *n receives the count.
 * Step indices are recorded modulo 2^32. */
int gcoreccd_read_collected(gcoreccd_t* h, float* xyz_um_host, uint32_t* step_host, uint64_t cap, uint64_t* n);

/* Coulomb field (eq. 6, V/cm) of the current snapshot, interleaved Ex,Ey,Ez in read_carriers order;
 * does not advance the simulation.  cap = number of carriers the buffer holds. */
int gcoreccd_eval_field(gcoreccd_t* h, float* Exyz_V_per_cm, uint64_t cap, int on_device);

/* ---- Batched independent events --------------------------------------------------
 * The paper's X-ray workload is many small clouds (N = E/3.77 eV holes per photon) whose
 * holes repel each other only inside their own event, and its GPU is under-utilised below ~1e3 holes
 * (PAPER.md:92).  A batch runs every event exactly as if it had been loaded alone into a fresh handle with the
 * same parameters (same eq. 6 sum over the event's own holes, same a2..a8, same Philox stream keyed by
 * (seed, carrier id, the EVENT's step index)), but all events advance concurrently: one warp (<= 32 holes), one
 * thread block, or - when there are few large events - one cluster of 2 or 4 thread blocks owns one event for its whole
 * life, with the state in registers / shared memory.  All events share the handle's image, counters and
 * pair_interactions (sum over events and steps of n_event^2).
 *
 * load_events: event e owns carriers [event_offsets[e], event_offsets[e+1]) of xyz_um (interleaved x,y,z FP32,
 *   host or device per on_device); event_offsets is a HOST array of n_events+1 non-decreasing entries starting
 *   at 0.  Carrier ids continue the handle's load order (id = n_loaded + index).  An event may be empty; none
 *   may exceed GCORECCD_EVENT_MAX_CARRIERS (CAPACITY; larger events belong in load_carriers), the total may not
 *   exceed max_carriers (CAPACITY).  Non-finite coordinates or z > thickness => INVALID, nothing loaded.
 *   Holes loaded at z <= z_well are collected when their event first runs.  STATE if the handle still holds
 *   drifting carriers (single event or an unfinished batch).  Replaces a finished batch.  Synchronous.
 * run_events: every unfinished event takes up to max_steps more steps (or runs to full collection).
 *   Synchronous.  Returns OK when every hole is collected, MAX_STEPS (+1) otherwise; *events_left and
 *   *carriers_left (host, may be NULL) receive what is still drifting.
 * get_events: per-event drifting holes and step index as of the last run_events (host arrays of cap_events
 *   entries, either may be NULL); *n_events receives the batch size.
 * read_event_carriers: the drifting holes of one event (stable load order), host buffers, either may be NULL. */
#define GCORECCD_EVENT_MAX_CARRIERS 4096
int gcoreccd_load_events(gcoreccd_t* h, const float* xyz_um, const uint64_t* event_offsets_host, uint64_t n_events,
                         int on_device);
int gcoreccd_run_events(gcoreccd_t* h, uint64_t max_steps, uint64_t* events_left, uint64_t* carriers_left);
int gcoreccd_get_events(gcoreccd_t* h, uint64_t* n_active_host, uint64_t* step_host, uint64_t cap_events,
                        uint64_t* n_events);
int gcoreccd_read_event_carriers(gcoreccd_t* h, uint64_t event, float* xyz_um_host, uint32_t* id_host, uint64_t cap,
                                 uint64_t* n);

/* ---- Workload front end ---------------------------------------------------------------
 * X-rays: a photo-electron of energy E_e makes N = E_e / w_e holes (w_e = 3.77 eV at 140 K),
 * initially a 3-D Gaussian cloud around the interaction point whose standard deviation depends on E_e (that model
 * is in the paper's references, not its text: sigma is an input here).
 *
 * xray_hole_count: floor(E_e_eV / w_eV); 0 if either is not positive.  Pure host arithmetic.
 * generate_cloud: draws n holes ~ N(centre, sigma^2 I) ON THE GPU and appends them exactly as load_carriers would
 *   (ids continue, z <= z_well collected at once).  Hole i uses generator index first_index + i: Box-Muller of
 *   Philox4x32-10(counter (index_lo, 'XRAY', index_hi, 0), key gen_seed), FP64, z above the back surface mirrored,
 *   rounded to FP32 — so chunked calls with consecutive indices equal one call.  centre_um: 3 host doubles.
 *   sigma_um >= 0.  Errors as load_carriers (INVALID also if the centre is outside (-inf, thickness]).
 * generate_xray_events: one batch of n_events independent clouds for run_events (replaces load_events):
 *   event e gets floor(E_e_eV[e] / w_eV) holes around centre_um[3e..3e+2] with sigma_um[e]; all arrays are HOST
 *   arrays; generator index = first_index + position of the hole in the batch.  counts_out (host, n_events entries,
 *   may be NULL) receives the hole count per event.  Errors as load_events.
 * load_carriers_file: text file, one hole per line "x y z" in um separated by blanks, tabs, commas or semicolons;
 *   empty lines and lines starting with '#' are skipped ("load the charge positions ... from an
 *   external file"; the paper does not give its format).  Appends like load_carriers; *n_read (host, may be NULL)
 *   receives the holes read.  INVALID on an unreadable file or a malformed line (nothing is loaded).
 * save_collected_file: writes "id x y z step" per collected hole, ascending id, with a '#' header line
 *   ("whether final results should be saved to a file"); *n_written may be NULL. */
uint64_t gcoreccd_xray_hole_count(double E_e_eV, double w_eV);
int gcoreccd_generate_cloud(gcoreccd_t* h, uint64_t n, const double* centre_um_host, double sigma_um, uint64_t gen_seed,
                            uint64_t first_index);
int gcoreccd_generate_xray_events(gcoreccd_t* h, uint64_t n_events, const double* E_e_eV_host, const double* centre_um_host,
                                  const double* sigma_um_host, double w_eV, uint64_t gen_seed, uint64_t first_index,
                                  uint64_t* counts_out_host);
int gcoreccd_load_carriers_file(gcoreccd_t* h, const char* path, uint64_t* n_read);
int gcoreccd_save_collected_file(gcoreccd_t* h, const char* path, uint64_t* n_written);

/* ---- Target sharding over several GPUs ---------------------------------------------
 * The fields of different targets j of eq. 6 are independent given all source positions, so the rows of
 * the interaction matrix shard over G GPUs: every rank holds the WHOLE active state (16 B per hole), rank g runs a1..a7
 * for the targets of its share against all sources, compacts its survivors (a8) into a MESSAGE, and the G messages
 * concatenated in rank order are the next step's state — in the same stable order one GPU would produce.  The share
 * of rank g is the contiguous 256-hole tiles [floor(g T/G), floor((g+1) T/G)) of the T = ceil(n_active/256) tiles: a
 * pure function of n_active, so shares re-balance every step without communication.  The only exchange per step is
 * the all-gather of the messages, which is the CALLER's plumbing (NCCL through torch.distributed, or peer-mapped
 * buffers); the library never waits on another rank inside a kernel.  Images, counters and collection records stay
 * rank-local: the global image is the integer sum over ranks, and sum_g pair_interactions_g = sum_steps n_active^2.
 *
 * set_shard: rank < world <= 64; only on an empty handle (before the first load / after reset); world = 1 restores
 *   the unsharded mode.  INVALID with GCORECCD_COULOMB_OFF (independent carriers: run replicas).  Every rank then
 *   loads the SAME carriers in the same order (load_carriers / generate_cloud / load_snapshot); holes collected at
 *   load are binned by rank 0 only.  While world > 1, step / run_to_collection / eval_field / profile_step return STATE.
 * shard_message_bytes: bytes a message buffer should have for the handle's current upper bound on n_active (refreshed
 *   by get_state): 256-byte header + 16 bytes x entries, entries = 256 x ceil(tiles/world) with tiles rounded up to a
 *   power of two.  Identical on all ranks that called get_state at the same step.
 * shard_local: a1..a7 for this rank's share + compaction of its survivors into msg_dev (DEVICE pointer, 16-byte
 *   aligned, msg_bytes as above or larger; layout header | x[] | y[] | z[] | id[]).  Asynchronous on the stream.
 *   Does not change the state.  CAPACITY if the buffer cannot hold the largest share.
 * shard_commit: msgs_host is a HOST array of `world` DEVICE pointers, message g produced by rank g for the SAME step
 *   with the SAME msg_bytes (slices of an all-gather receive buffer, or the ranks' own buffers mapped through CUDA
 *   IPC / symmetric memory: the loads then cross NVLink inside this kernel).  Replaces the active state by the
 *   concatenation, step += 1, pair_interactions += share x n_active, plans the next share.  Asynchronous.  A message
 *   whose (n_active, step, rank) header disagrees with this rank sets a sticky flag that get_state reports as STATE.
 *   The caller must not overwrite a message before every rank has committed it (alternate two buffers). */
int gcoreccd_set_shard(gcoreccd_t* h, uint32_t rank, uint32_t world);
uint64_t gcoreccd_shard_message_bytes(gcoreccd_t* h);
int gcoreccd_shard_local(gcoreccd_t* h, void* msg_dev, uint64_t msg_bytes);
int gcoreccd_shard_commit(gcoreccd_t* h, const void* const* msgs_host, uint32_t n_msgs, uint64_t msg_bytes);
/* Peer-mapped messages (CUDA IPC / symmetric memory: msgs_host[g] points INTO rank g's own buffer): with on != 0 the
 * commit kernel itself waits, message by message, until the header of THIS step has arrived (a 64-bit word written
 * last, release at system scope, by shard_local: (epoch << 32) | step + 1, epoch changing at every reset / set_shard),
 * so no barrier between shard_local and shard_commit is needed.  Requires two message buffers used alternately and
 * ranks that really run at the same time on different GPUs; never set it when the messages of a step are produced
 * AFTER the commit is enqueued on the same device (the kernel would wait forever).  Default off. */
int gcoreccd_set_shard_wait(gcoreccd_t* h, int on);

/* ---- Far-field approximation of eq. 6 — a VARIANT, off by default --------------------------
 * The exact path sums all N_a^2 ordered pairs.  With set_farfield(theta >= 0) step a1 is replaced by
 * a treecode: the active holes are kept in Hilbert-curve order (re-sorted every resort_every field evaluations; 0 => every
 * 2nd for the first 192 evaluations after set_farfield / reset, while the cloud is dense, then every 4th), an
 * implicit 8-ary tree of runs of 8*8^l consecutive holes carries, per node, its hole count m, centre of charge c and the
 * radius a of the ball about c holding its members; every group of 256 consecutive targets replaces a node by ONE
 * pseudo-hole of charge m at c when  a <= theta * |x_t - c|  holds for every target t of the group, and sums all other
 * holes exactly.  a2..a8 are unchanged.
 * Stated bound (monopole about the centre of charge; the dipole vanishes): for every target j
 *     |E_approx,j - E_exact,j|  <=  B(theta) * sum_{accepted nodes} m K' / d_j^2 ,   B = theta^2 (3 - 2 theta)/(1 - theta)^2,
 * d_j the distance from j to the node's centre; the near field is exact; theta = 0 accepts no node (exact sum in
 * another order).  Measured errors are one to two orders below the bound (tests/test_gpu_farfield.py).
 * Consequences: the active set is no longer in load order (read_carriers / eval_field return the current curve order;
 * match by id); pair_interactions still counts N_a^2 per step (the pairs REPRESENTED) — the interactions actually
 * evaluated are in farfield_stats and no throughput claim of the exact metric may use this variant.
 * set_farfield: theta in [0, 1) switches the variant on, theta < 0 off.  Synchronises.  On a sharded handle every rank
 *   must make the same call at the same step: the re-sort and the tree are then computed identically on every rank
 *   (replicated state) and only the walk is sharded, each rank walking the groups of its own share.
 *   While fewer than min_active holes are drifting (0 => 24,576; 1 => never) the all-pairs kernel is used instead:
 *   below a few 1e4 holes it is the faster of the two (measured), and it is exact.
 * farfield_stats: interactions evaluated since set_farfield — pseudo-hole (far) and exact (near), each counted per
 *   target — and B(theta).  Host pointers, any may be NULL.  STATE if the variant is off. */
int gcoreccd_set_farfield(gcoreccd_t* h, double theta, uint32_t resort_every, uint64_t min_active);
int gcoreccd_farfield_stats(gcoreccd_t* h, uint64_t* far_evals, uint64_t* near_evals, double* bound_B);

/* Run ONE step as two launches with CUDA events between them (on the handle's stream) and return the device time of
 * each in milliseconds: ms[0] field (a1), ms[1] advance (a2..a8: update, collection, in-place compaction), ms[2] = 0
 * (compaction was a kernel of its own in version 0.1), ms[3] whole step.  Synchronous. */
int gcoreccd_profile_step(gcoreccd_t* h, float ms_host[4]);

/* Small populations (below ~1e3 charges "the GPU is subutilised"): while the handle's upper bound on
 * n_active is <= max_active, gcoreccd_step / run_to_collection run all their steps in ONE cooperative launch of a
 * persistent kernel (field -> grid barrier -> a2..a8 -> grid barrier per step) instead of two launches per step.
 * Up to 32 targets per SM (2,368 / 4,736 holes on 148 SMs) a warp owns its 2 / 4 targets for the whole step and a
 * step costs ONE grid barrier (gc_persist_warp.cuh); run_to_collection lets a launch end when the population has decayed
 * into the range of a smaller variant and continues with that one.
 * on = 0 turns the persistent path off, on = 2 keeps it but without the warp-owner kernels (tuning / test hooks);
 * max_active = 0 keeps the default (24,576).  Same physics, same Philox
 * counters; the FP32 summation order of eq. 6 differs between the two paths, nothing else.  All-pairs, unsharded
 * handles only (otherwise ignored). */
int gcoreccd_set_persistent(gcoreccd_t* h, int on, uint64_t max_active);

/* Number of kernels this handle has launched so far (bench.py's gpu_launches). */
uint64_t gcoreccd_kernel_launches(gcoreccd_t* h);

/* Normal triple of (seed, id, step) as the integrator draws it (test hook for the Philox stream, a5). */
int gcoreccd_debug_normals(gcoreccd_t* h, const uint32_t* id_host, const uint64_t* step_host, uint64_t n,
                           double* n_xyz_host, uint32_t* words_host);

/* Hole mobility of eq. 2 at n field magnitudes E (V/cm, host pointers) as the kernels evaluate it — piecewise
 * degree-8 interpolants of (1 + (E/Ec)^beta)^(-1/beta) tabulated at create, relative error < 1e-15 — and by the direct
 * exp/log form (test hook for a3; cm^2 / (V s)). */
int gcoreccd_debug_mobility(gcoreccd_t* h, const double* E_host, uint64_t n, double* mu_table_host, double* mu_direct_host);

/* The same table built and evaluated ON THE HOST (no GPU needed) for temperature T_K: lets the CPU test suite check the
 * interpolants against an independent evaluation of eq. 2. */
int gcoreccd_mobility_table_host(double T_K, const double* E_host, uint64_t n, double* mu_host);

/* Instruction-throughput probe (no handle; current device): runs `iters` x 32 instructions of one kind on one SM with
 * `warps_per_subpartition` (1..4) warps per SM sub-partition and returns the cycles per warp-instruction per
 * sub-partition.  Kinds: 0 FFMA2 three distinct operands, 1 FFMA2 a*a+c, 2 FFMA2 one operand shared by consecutive
 * instructions, 3 FADD2, 4 FMUL2, 5 scalar FFMA three distinct, 6 scalar FFMA shared operand, 7 DFMA, 8 MUFU.RSQ,
 * 9 the 11 packed instructions + 2 MUFU of one eq. 6 interaction pair (per packed instruction), 10 F2F f64->f32,
 * 11 F2F f32->f64, 12 DADD, 13 one eq. 6 interaction per lane on the FP64 pipe, 14-16 the FP32 mix on 8 packs with
 * 1 / 2 / 4 FP64-pipe targets interleaved (cycles per round of 8 packs).  The evidence behind
 * DESIGN.md 6.1 / 6.8 (`python bench.py --microbench`); not on the hot path. */
int gcoreccd_debug_microbench(int kind, uint32_t iters, uint32_t warps_per_subpartition, double* cycles_per_inst_host);

/* ---- Allocation-free entry point ---------------------------------------------------------------------------------
 * Some callers cannot call cudaMalloc: code under CUDA-graph capture, tight serving loops, harnesses that forbid it.
 * gcoreccd_field_noalloc evaluates the Coulomb field of eq. 6 (the operation of gcoreccd_eval_field) for
 * n <= GCORECCD_NOALLOC_MAX_CARRIERS holes WITHOUT a handle and without allocating anything: no cudaMalloc, cudaFree or
 * allocating library routine is called, here or at set-up.  Its scratch (positions as structure of arrays, the work
 * plan, the partial-sum planes: 6,488,320 bytes) is a file-scope `static __device__` array inside the library, which
 * every GPU that loads the library therefore holds until the process exits.
 *   xyz_um_dev  DEVICE pointer, n interleaved (x, y, z) in um, FP32 (layout of gcoreccd_load_carriers); caller-owned,
 *               read only; not validated (a non-finite coordinate gives non-finite fields)
 *   softening_um, eps_si   as in gcoreccd_params (eps_si = 0 -> 11.7; softening 0 evaluates eq. 5, R5)
 *   Exyz_dev    DEVICE pointer, receives n interleaved (Ex, Ey, Ez) in V/cm, same order as the input; caller-owned
 *   stream      cudaStream_t the four kernels are enqueued on (NULL = default stream); the call does NOT synchronise
 * Runs on the CURRENT device (sm_100 required: GCORECCD_ERR_CUDA otherwise, no fallback).  The first call on a device
 * looks the array's address up (cudaGetSymbolAddress); nothing else is kept between calls.
 * Returns GCORECCD_ERR_CAPACITY for n > GCORECCD_NOALLOC_MAX_CARRIERS, GCORECCD_ERR_INVALID for null pointers or a
 * negative / non-finite parameter; n = 0 is a no-op.  gcoreccd_field_noalloc_error() gives the detail of the calling
 * thread's last failure ("" if none).
 * ALL calls share the one array, on every stream and from every thread: two calls whose kernels overlap on the GPU
 * race on it (undefined results).  Keep them on one stream, or order them with events.  The array keeps the last call's
 * contents; each call re-initialises what it reads. */
#define GCORECCD_NOALLOC_MAX_CARRIERS 16384u
int gcoreccd_field_noalloc(const float* xyz_um_dev, uint64_t n, double softening_um, double eps_si, float* Exyz_dev,
                           void* stream);
const char* gcoreccd_field_noalloc_error(void);

const char* gcoreccd_strerror(int code);
const char* gcoreccd_last_error(gcoreccd_t* h);   /* detail of the last failure on this handle ("" if none) */
const char* gcoreccd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GCORECCD_H */
