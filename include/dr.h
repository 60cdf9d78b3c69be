/* dr.h — C-ABI of the B200-native Diffusion Restore hot path (arXiv 2605.08916).
 *
 * The per-frame step of N independent Markov chains in primary sample space (PSS):
 * Alg. 1 Initialize/Accumulate, Alg. 2 Evolve (L530-L543),
 * Alg. 3 Resolve (L545-L550), Alg. 4 LocalDynamics (L707-L723), for the five samplers of
 * L733-L747.  Readings of everything the paper leaves open: DESIGN.md section 2 (Q1-Q20).
 *
 * Conventions
 *  - plain C, no exceptions cross this boundary; every call returns a dr_status
 *    (negative = failure and no state change where possible, positive = warning);
 *    dr_last_error() gives a thread-local message for the last non-OK status.
 *  - "host" / "dev" in a parameter name says where the pointer lives.  Host arrays given to
 *    dr_scene_create* are copied (the caller may free them on return).  Chain state, the
 *    accumulation buffer and the output image are CALLER-OWNED DEVICE MEMORY (e.g. torch
 *    tensors); the library never frees them and they must outlive the dr_chains handle.
 *  - `stream` is a cudaStream_t passed as void* (NULL = default stream).  All work is
 *    asynchronous on that stream; only dr_chains_stats, dr_profile_*, dr_chains_work_stats and the
 *    *_download / *_upload hooks synchronise it.
 *  - one GPU (the current device), fp32 arithmetic, sm_100a only, no CPU fallback.
 */
#ifndef DR_H_
#define DR_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  DR_OK = 0,
  DR_WARN_NO_TOURS = 1,      /* dr_chains_stats: a resolve ran before any tour completed: zero image, no division */
  DR_ERR_INVALID_ARG = -1,
  DR_ERR_UNSUPPORTED = -2,
  DR_ERR_CUDA = -3,
  DR_ERR_NONFINITE = -4,     /* non-finite value in host input */
  DR_ERR_OOM = -5
} dr_status;

/* the five samplers. */
typedef enum {
  DR_METROPOLIS = 0,
  DR_MALA = 1,
  DR_METROPOLIS_RESTORE = 2,
  DR_MALA_RESTORE = 3,
  DR_DIFFUSION_RESTORE = 4,
  DR_PATH_TRACING = 5        /* ordinary path tracing on the same buffers, the baseline of its section 6:
                                every chain is drawn anew each iteration, f accumulated with unit weight */
} dr_method;

/* pbrt-v4 diffuse / dielectric / conductor + DiffuseAreaLight, simplified as in DESIGN.md Q6-Q7. */
typedef enum { DR_MAT_LAMBERT = 0, DR_MAT_DIELECTRIC = 1, DR_MAT_GGX_CONDUCTOR = 2, DR_MAT_EMITTER = 3 } dr_mat_kind;

typedef struct {
  int32_t kind;             /* dr_mat_kind */
  float albedo_or_f0[3];    /* Lambert albedo or conductor F0 */
  float ior;                /* dielectric: inside / outside index ratio (> 0) */
  float roughness;          /* GGX alpha in (0, 1] */
  float emission[3];        /* emitter radiance on the front face (geometric normal side) */
} dr_material;

typedef struct {
  const float* host_vertices;       /* 3 * nv */
  uint32_t nv;
  const uint32_t* host_indices;     /* 3 * nt, counter-clockwise = front */
  uint32_t nt;
  const uint32_t* host_tri_material;/* nt, index into materials */
  const dr_material* host_materials;
  uint32_t nm;
  float env_radiance[3];            /* radiance of rays that escape */
  float cam_pos[3], cam_look[3], cam_up[3];
  float vfov_deg;                   /* pinhole camera, vertical field of view */
  uint32_t width, height;           /* image W x H; pixel map DESIGN.md Q4 */
  uint32_t max_path_len;            /* L segments, PSS dimension d = 2L (Q5); 1 <= L <= 16 */
  uint32_t nee;                     /* 0 / 1: next-event estimation + MIS (Q21): emitters sampled by area
                                       at every Lambert / GGX vertex, balance heuristic; four coordinates per vertex, d = 4L */
} dr_scene_desc;

/* 2-D analytic target (d = 2): mixture of wrapped Gaussians, f = (p,p,p), closed-form score.
 * Exercises the samplers without ray tracing (stationarity tests). */
typedef struct {
  uint32_t n_components;            /* 1..16 */
  const float* host_weights;        /* n */
  const float* host_means;          /* 2 n */
  const float* host_stddevs;        /* n */
  uint32_t width, height;
} dr_analytic2d_desc;

typedef struct {
  int32_t method;            /* dr_method */
  uint32_t n_chains;         /* N = dispatchCount */
  float stddev;              /* L747: 1e-2 Metropolis*, 5e-3 Langevin-based; > 0 */
  float c_tilde;             /* rotation strength c~ = dt c / 2 (L700), Diffusion Restore only; >= 0 */
  float dt;                  /* L755: 1e-5; holding rate lambda = 1/dt (L659), Diffusion Restore only; > 0 */
  float m;                   /* L754: expected local steps per tour, kappa0 = p_lambda / (m dt) (L752); > 0 */
  float large_step_prob;     /* L747: 0.3 for plain Metropolis / MALA; ignored by Restore variants; in [0,1] */
  float p_lambda_override;   /* > 0: use as p_lambda; <= 0: bootstrap from the init states (DESIGN.md a0) */
  uint64_t seed;             /* Philox key (Q14) */
  uint32_t chain_offset;     /* global id of chain 0: RNG streams are keyed by global chain id, so a run sharded
                                over several GPUs draws the same numbers as the unsharded run */
  uint32_t rao_blackwell;    /* Restore variants, 0 / 1: accumulate E[dtau | x] = 1 / (lambda + kappa) instead of the sampled
                                dtau (Rao-Blackwellised holding time); the kill decision stays the race */
  uint32_t a_mode;           /* antisymmetric part of the Langevin drift (future work L822): 0 = the paper's
                                diag(A_block), coordinate pairs (2i, 2i+1); 1 = pairs (4i, 4i+2) and (4i+1, 4i+3) (Q24) */
  uint32_t rho_grid;         /* regeneration density rho (future work L824): 0 = uniform; G in 1..64:
                                piecewise constant on a G x G tiling of the film coordinates (x0, x1), uniform in the others;
                                the killing rate becomes (rho / rho_lambda) kappa0 / p_hat.  Plain Metropolis / MALA never regenerate:
                                for them rho only sets where the chains START (dr_chains_init draws x ~ rho and the bootstrap of
                                p_lambda divides by rho); their stationary law is unchanged.  DR_PATH_TRACING averages its samples
                                with unit weight, so a non-uniform draw would bias it: rho_grid != 0 is DR_ERR_INVALID_ARG there */
  const float* host_rho;     /* G*G tile probabilities, row-major (tile = ty * G + tx), > 0, summing to one (copied) */
} dr_config;

/* The paper's parameters for `method`, for C callers and the binding alike: zeroes *host_out, then sets method and
 *   stddev           1e-2 for Metropolis and Metropolis-Restore, 5e-3 for the Langevin-based samplers; a stddev
 *                    argument > 0 replaces it
 *   large_step_prob  0.3 for plain Metropolis / MALA, 0 otherwise (L747)
 *   dt = 1e-5 (L755), m = 64 (L754)
 *   c_tilde          stddev^2 / 2 of the stddev in use: this build's default rotation strength (Q10; the paper gives none)
 * n_chains, seed and the other fields stay zero for the caller to fill in.  DR_ERR_INVALID_ARG for an unknown method, a null
 * pointer or a stddev that is not finite. */
dr_status dr_config_default(int32_t method, double stddev, dr_config* host_out);

typedef struct {
  uint64_t tours;            /* tourCount */
  uint64_t mutations;        /* Accumulate calls = chain-iterations, init included */
  uint64_t rays;             /* closest-hit queries */
  uint64_t mh_accepts;       /* accepted Metropolis-Hastings proposals */
  uint64_t nonfinite;        /* evaluations with non-finite f or score (treated as p = 0, Q18) */
  uint32_t kills_last_step;  /* == regen_queue_len */
  uint32_t regen_queue_len;
  uint32_t iteration;        /* n of the last completed iteration (0 = init) */
  float p_lambda, kappa0, lambda;
  uint32_t no_tour_resolves; /* resolves since init that found tourCount == 0 and wrote a zero image */
  uint32_t wave_timeouts;    /* evaluations ended by k_wave's watchdog (never, unless the queue protocol is broken): dr_chains_stats
                                then returns DR_ERR_CUDA instead of letting a kernel spin on the GPU for ever */
  uint64_t grad_states;      /* evaluations that ran the reverse pass for the score (states with a non-zero score, a6) */
  uint64_t lit_init;         /* init states with p > 0: lit_init / N = fraction of uniform PSS samples that contribute */
} dr_stats;

typedef struct {
  uint32_t n_tris, n_nodes, depth, smem_nodes; /* BVH8 nodes, tree depth; smem_nodes is always 0 (no node staging: the field keeps the layout) */
  float sah_cost;
  float eps_ray;
  size_t device_bytes;
} dr_scene_info;

typedef struct dr_scene dr_scene;   /* opaque */
typedef struct dr_chains dr_chains; /* opaque */

const char* dr_last_error(void);

/* Validates the description (finite vertices, indices < nv, materials in range, 1 <= L <= 16, W,H >= 1),
 * builds a SAH BVH2 on the host, collapses it to a BVH8, uploads.  The scene owns its device memory. */
dr_status dr_scene_create(const dr_scene_desc* desc, dr_scene** out);
dr_status dr_scene_create_analytic2d(const dr_analytic2d_desc* desc, dr_scene** out);
dr_status dr_scene_destroy(dr_scene* scene);
dr_status dr_scene_get_info(const dr_scene* scene, dr_scene_info* host_out);

/* Bytes of device memory dr_chains_create needs for N chains on this scene (256-byte aligned). */
size_t dr_chains_state_bytes(const dr_scene* scene, const dr_config* cfg);

/* Validates cfg (stddev > 0, dt > 0, m > 0, probabilities in [0,1], N >= 1) and lays the chain state out in
 * dev_state (SoA planes).  dev_accum_rgba: W*H float4 (RGB = sum w f/p_hat, A = sum w/p_hat). */
dr_status dr_chains_create(const dr_scene* scene, const dr_config* cfg, void* dev_state, size_t state_bytes,
                           float* dev_accum_rgba, dr_chains** out);
dr_status dr_chains_destroy(dr_chains* chains);

/* Alg. 1 for every chain (+ bootstrap of p_lambda and kappa0): zeroes the accumulation buffer and counters,
 * x ~ U[0,1)^d keyed by (chain, iteration 0, frame_index), evaluate, Accumulate. */
dr_status dr_chains_init(dr_chains* chains, uint32_t frame_index, void* stream);

/* Alg. 2 for every chain, `iterations` times.  `method` must equal the method the chains were created with
 * (DR_ERR_INVALID_ARG otherwise). */
dr_status dr_step(dr_chains* chains, int32_t method, uint32_t iterations, void* stream);

/* Alg. 3: dev_rgb_out[W*H*3] = N_pix * kappa0 / tourCount * accum (Restore), N_pix * p_lambda / N_mut * accum (plain MH)
 * or N_pix / N_mut * accum (path tracing).  Asynchronous: if tourCount == 0 the kernel writes zeros (no division) and counts the event in
 * dr_stats.no_tour_resolves; the next dr_chains_stats then returns DR_WARN_NO_TOURS. */
dr_status dr_resolve_image(dr_chains* chains, float* dev_rgb_out, void* stream);

/* Alg. 3 for a run sharded over several GPUs: dev_accum_sum is the all-reduced accumulation buffer
 * (W*H float4), tours_total / mutations_total the all-reduced counters (mutations_total > 0).  p_lambda and kappa0
 * are this shard's; they are identical on every shard when p_lambda_override is used.  Asynchronous; tours_total == 0
 * is handled as in dr_resolve_image. */
dr_status dr_resolve_image_sharded(dr_chains* chains, const float* dev_accum_sum, uint64_t tours_total,
                                   uint64_t mutations_total, float* dev_rgb_out, void* stream);

/* The same with ONE collective and no host synchronisation per frame: dr_pack_frame writes dr_frame_floats(chains) =
 * W*H*4 + 8 floats into dev_buf (16-byte aligned): this shard's accumulation buffer followed by tourCount and the mutation
 * count as four 16-bit limbs each, stored as floats, so that an fp32 all-reduce(sum) over up to 256 shards adds them exactly;
 * dr_resolve_image_packed takes the all-reduced buffer.  Both asynchronous. */
size_t dr_frame_floats(const dr_chains* chains);
dr_status dr_pack_frame(dr_chains* chains, float* dev_buf, void* stream);
dr_status dr_resolve_image_packed(dr_chains* chains, const float* dev_buf_sum, float* dev_rgb_out, void* stream);

/* Per-kernel timing with CUDA events on the caller's stream (bench.py's roofline).  dr_profile_enable(on) resets
 * the totals; while on, every kernel launch of dr_chains_init / dr_step / dr_resolve_image* is bracketed by two
 * events.  dr_profile_read synchronises the stream and returns, per kernel class, the summed device time in ms and
 * the number of launches (arrays of DR_PROF_COUNT entries). */
enum { DR_PROF_PROPOSE = 0, DR_PROF_RAYGEN = 1, DR_PROF_TRACE = 2, DR_PROF_SHADE = 3, DR_PROF_GRAD = 4, DR_PROF_DECIDE = 5,
       DR_PROF_SCAN = 6, DR_PROF_SCATTER = 7, DR_PROF_RESOLVE = 8, DR_PROF_COUNT = 9 };
dr_status dr_profile_enable(dr_chains* chains, int32_t on, void* stream);
dr_status dr_profile_read(dr_chains* chains, double* host_ms, uint64_t* host_launches, void* stream);
/* Work of the last evaluation launch: host_out3 = {rays, BVH8 node visits, triangle tests} of the chains' last
 * proposals (re-evaluated with counters; values only).  Synchronises. */
dr_status dr_chains_work_stats(dr_chains* chains, uint64_t* host_out3, void* stream);

/* Synchronises the stream and copies the counters.  DR_WARN_NO_TOURS (with host_out filled) if no_tour_resolves != 0. */
dr_status dr_chains_stats(dr_chains* chains, dr_stats* host_out, void* stream);

/* ---- test hooks (parity harness; same library) ---------------------------------------------------------- */
/* Host arrays, row-major: x[N*d], score[N*d], p[N], f_over_p[N*3], pix[N], killed[N], sig[N] (hash of the
 * discrete decisions of the state's path).  Any output pointer may be NULL. */
dr_status dr_chains_download(dr_chains* chains, float* host_x, float* host_p, float* host_f_over_p, uint32_t* host_pix,
                             uint8_t* host_killed, float* host_score, uint32_t* host_sig, void* stream);
/* Teacher forcing: overwrite the state (host_sig may be NULL) and set the iteration counter; rebuilds the
 * regeneration queue. */
dr_status dr_chains_upload(dr_chains* chains, const float* host_x, const float* host_p, const float* host_f_over_p,
                           const uint32_t* host_pix, const uint8_t* host_killed, const float* host_score,
                           const uint32_t* host_sig, uint32_t iteration, void* stream);
/* Per-chain record of the last iteration: accepted flag and sampled weight (dtau, or 1 for plain MH). */
dr_status dr_chains_last_step(dr_chains* chains, uint8_t* host_accepted, float* host_weight, void* stream);
/* Killed chain ids in ascending order; host_ids may be NULL to query the length. */
dr_status dr_regen_queue_download(dr_chains* chains, uint32_t* host_ids, uint32_t* host_len, void* stream);
/* Closest hit for n rays (device arrays o[3n], d[3n] -> t[n] (-1 = miss), prim[n] (0xFFFFFFFF = miss)). */
dr_status dr_trace_rays(const dr_scene* scene, const float* dev_o, const float* dev_d, uint32_t n, float* dev_t,
                        uint32_t* dev_prim, void* stream);
/* dr_trace_rays for callers that must not allocate device memory at the time of the call.
 *
 * Who that is: code running where cudaMalloc / cudaFree are forbidden or harmful.  Examples: a real-time frame loop or a
 * serving process with a fixed memory budget, where an allocation can fail late or stall (cudaFree waits for the whole
 * device); a host program that has handed all of the GPU's memory to its own pool and leaves nothing for the driver; a
 * plugin that lives inside someone else's process and is not allowed to change that process's memory footprint.
 * dr_trace_rays takes its ray queue, hit records and queue counters (40 bytes per ray + 8) from cudaMalloc on every call
 * and waits for the stream before it frees them.  This variant runs the SAME kernels on the same inputs and writes the same
 * outputs (bit for bit), but its scratch is a fixed array that is part of the library image:
 *   - the array holds DR_TRACE_NOALLOC_MAX_RAYS rays (40 bytes each + 256): about 2.5 MiB, present on every GPU that
 *     loads the library from the moment it is loaded until the process exits, whether this call is used or not;
 *   - n > DR_TRACE_NOALLOC_MAX_RAYS is refused with DR_ERR_INVALID_ARG and nothing is launched: split the batch;
 *   - the call makes no cudaMalloc, cudaFree or other allocating call, and does not synchronise: the work is queued on
 *     `stream` like every other asynchronous call of this header.  dev_o, dev_d, dev_t, dev_prim are the caller's,
 *     as for dr_trace_rays;
 *   - the FIRST call on each device looks up the array's device address (a cudaGetSymbolAddress, once per device,
 *     with the scene's device current as for every call here).  Make that first call during set-up, before the
 *     stream is put into capture mode;
 *   - every call on a device uses the one array, and the array keeps what the last call left in it.  The call clears
 *     the two queue counters it needs at zero itself.  Two calls whose GPU work can overlap (different streams without an
 *     event between them, or two host threads) race on the array and give wrong hits: keep the calls of one device on one
 *     stream, or order them with events. */
#define DR_TRACE_NOALLOC_MAX_RAYS 65536u
dr_status dr_trace_rays_noalloc(const dr_scene* scene, const float* dev_o, const float* dev_d, uint32_t n, float* dev_t,
                                uint32_t* dev_prim, void* stream);
/* Target evaluation for n states (device arrays, row-major x[n*d]) -> f[3n], p[n], pix[n], score[n*d] (if
 * non-NULL), nrays[n], sig[n]. */
dr_status dr_eval_states(const dr_scene* scene, const float* dev_x, uint32_t n, float* dev_f, float* dev_p,
                         uint32_t* dev_pix, float* dev_score, uint32_t* dev_nrays, uint32_t* dev_sig, void* stream);
/* The same, choosing the form of rows a3-a5 (identical results, state by state): 0 = default, 1 = one k_trace + k_shade
 * launch per segment, 2 = one persistent k_wave launch (csrc/dr_wave.cuh) in the block shape the default would take for n
 * states, 3 / 4 = k_wave in its small / big block shape (640 threads with two triangle slots per lane below 400 000
 * states -- 160 000 with next-event estimation --, 768 threads with one above: csrc/dr_eval.cuh).  dr_chains_set_eval_form does the same for the evaluations inside
 * dr_chains_init / dr_step. */
dr_status dr_eval_states_form(const dr_scene* scene, const float* dev_x, uint32_t n, float* dev_f, float* dev_p,
                              uint32_t* dev_pix, float* dev_score, uint32_t* dev_nrays, uint32_t* dev_sig, int32_t form,
                              void* stream);
dr_status dr_chains_set_eval_form(dr_chains* chains, int32_t form);
/* Work statistics for n states (device x[n*d], values only): dev_out3[0..2] += {rays, BVH8 node visits, triangle
 * tests}.  bench.py derives the algorithmic FLOPs per ray of its roofline from these. */
dr_status dr_eval_work_stats(const dr_scene* scene, const float* dev_x, uint32_t n, uint64_t* dev_out3, void* stream);
/* Appendix C of the paper: the field b = L^* p_hat / p_hat that controls the bias of the
 * modified killing rate, for the Alg. 4 dynamics (step width stddev, rotation c_tilde, holding rate 1 / dt) on a 2-D analytic
 * scene.  dev_out[iy * G + ix] (double) = b at the centre of cell (ix, iy) of a G x G grid; the integral over the torus is a
 * midpoint rule on M x M points, in double (the difference cancels to O(dt)).  Analysis only: not part of dr_step.  Synchronises. */
dr_status dr_bias_field(const dr_scene* scene, double stddev, double c_tilde, double dt, uint32_t G, uint32_t M, double* dev_out,
                        void* stream);
/* Raw Philox blocks for n counters (device arrays ctr[4n] -> out[4n]) under key (seed lo, hi), and the stream
 * transforms of DESIGN.md Q14 for n words pairs: out[4n] = u[0,1), u(0,1], Box-Muller z0, z1. */
dr_status dr_philox_blocks(uint64_t seed, const uint32_t* dev_ctr, uint32_t n, uint32_t* dev_out, void* stream);
dr_status dr_rng_transforms(const uint32_t* dev_words, uint32_t n, float* dev_out, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* DR_H_ */
