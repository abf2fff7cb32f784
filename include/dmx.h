/* dmx.h — C-ABI of the B200-native DiffMJX hot path (arxiv 2506.14186).
 *
 * Batched adaptive-step rollouts of a MuJoCo-style penalty-contact rigid-body simulator over
 * independent environments, and the reverse-mode gradient of a terminal loss through the
 * accepted steps with Contacts From Distance (CFD) applied only in the backward pass.
 * Every step of the path runs in hand-written CUDA kernels (sm_100a); there is no CPU fallback.
 *
 * Conventions
 *   - "host" / "device" says where a pointer must live.  All device buffers and the CUDA
 *     stream are owned by the caller; the library owns only the dmx_model.
 *   - Batched arrays are env-major and row-contiguous.  Element type `real` is double for a
 *     model created with precision 64 and float for precision 32 (x0, ctrl, params, xT, dLd*,
 *     tape); h_replay and all statistics are always double / int.
 *   - State x = [q | v]: q[nq] (free joint: 3 position + unit quaternion
 *     w,x,y,z; hinge / slide: one scalar), v[nv] (free joint: world linear, body angular).
 *   - Calls only enqueue work on `cuda_stream`; they do not synchronise and do not allocate (all
 *     scratch is sized at dmx_model_create).  Calls on one model may be issued on different
 *     streams: each call takes its own work-queue counter (up to 64 calls in flight), and a reverse
 *     sweep waits (cudaStreamWaitEvent) for the previous reverse sweep of the same model, whose
 *     adjoint scratch it reuses.  dmx_model_set_tape_stages must not change between the rollout
 *     that writes a tape and the sweep that reads it; the tape records its layout and a sweep over
 *     a tape of another layout, batch size or plan returns zero gradients.
 *   - Return value: 0 ok; <0 invalid argument / CUDA error (text via dmx_last_error()).
 *     Numerical trouble inside one environment never fails a call, it is reported in
 *     stats.status[e]: 0 ok, 1 step budget exceeded, 2 step-size
 *     underflow, 3 non-finite, 4 tape full.  A failed environment returns its last accepted
 *     state and zero gradients.
 */
#ifndef DMX_H
#define DMX_H
#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { DMX_JNT_FREE = 0, DMX_JNT_HINGE = 1, DMX_JNT_SLIDE = 2 };
enum { DMX_GEOM_PLANE = 0, DMX_GEOM_SPHERE = 1, DMX_GEOM_CAPSULE = 2, DMX_GEOM_BOX = 3 };
enum { DMX_ACT_MOTOR = 0, DMX_ACT_PD = 1 };
enum { DMX_DOPRI5 = 0, DMX_TSIT5 = 1 };

typedef struct dmx_model dmx_model; /* opaque; owns device copies of the constants */

/* Model description: flattened kinematic tree, geoms, solref/solimp, friction
 * (BASELINE.json north_star; PAPER.md:41-45 state and dynamics, :51 collision, :58-68 Eq. 3,
 * impedance and regulariser).  All pointers are HOST pointers, copied at create.
 * Restrictions: body 0 is the world; body_parent[b] < b; at most one joint per body; free
 * joints only on children of the world; planes on the world body and first in a pair;
 * supported pairs: plane-sphere, plane-capsule (two end caps), plane-box (eight corners),
 * sphere-sphere (north_star subsystem 2). */
typedef struct {
  int nbody, njnt, nq, nv, nu, ngeom, npair;
  const int *body_parent;                                   /* [nbody]                        */
  const double *body_pos, *body_quat;                       /* [nbody*3], [nbody*4] in parent  */
  const double *body_mass;                                  /* [nbody]                        */
  const double *body_ipos, *body_iquat;                     /* inertial frame in the body     */
  const double *body_inertia_unit;                          /* [nbody*3] principal inertia per unit mass */
  const int *jnt_type, *jnt_body, *jnt_qadr, *jnt_vadr;     /* [njnt]                         */
  const double *jnt_axis, *jnt_pos;                         /* [njnt*3] in the body frame      */
  const double *jnt_damping, *jnt_armature;                 /* [njnt]                         */
  const int *geom_type, *geom_body;                         /* [ngeom]                        */
  const double *geom_size, *geom_pos, *geom_quat;           /* [ngeom*3], [ngeom*3], [ngeom*4] */
  const int *pair_geom1, *pair_geom2, *pair_condim;         /* [npair]; condim 1 or 3 (pyramidal) */
  const double *pair_friction;                              /* [npair]                        */
  const double *pair_solref;                                /* [npair*2] (timeconst, dampratio), Eq. 3 */
  const double *pair_solimp;                                /* [npair*5] (d_o,d_w,w,mid,power) */
  const double *pair_solimp_cfd;                            /* [npair*5] (d_c,d_0,w_c,m_c,p_c) */
  const double *pair_cfd_beta;                              /* [npair] softplus sharpness */
  const int *act_type, *act_jnt;                            /* [nu]                           */
  const double *act_gear, *act_kp, *act_kd;                 /* [nu]                           */
  double gravity[3];
  int newton_iters, ls_iters;                               /* fixed iteration scheme */
  const double *qpos0;                                      /* [nq] reference pose for the diagonal approximation
                                                               A^ of J M^-1 J^T   */
} dmx_model_desc;

/* Adaptive embedded Runge-Kutta options (Tsit5 / Dopri5 and the PID controller
 * with P=0.2, I=0.4, D=0 at PAPER.md:347). */
typedef struct {
  int tableau;          /* DMX_DOPRI5 | DMX_TSIT5 */
  double rtol, atol;    /* error = sqrt(mean((e_j / (atol + rtol*max(|y_n|,|y_n+1|)_j))^2)), accept iff <= 1 */
  double h0;            /* initial step proposal */
  double pcoeff, icoeff, safety, fac_min, fac_max;
  int max_steps;        /* budget of attempted steps per environment */
} dmx_solver_opts;

/* Per-environment step statistics; DEVICE pointers, each [nenv]; any may be NULL.
 * n_newton_unconverged: F evaluations of the forward pass whose fixed-iteration Newton solve did not
 * end on a full step inside an unchanged active set.  n_newton_unconverged_bwd: the same count over the contact solves
 * of the reverse sweep (F~ with cfd_on, or F when the stages are recomputed); the vector-Jacobian product of such a stage
 * is the implicit-function gradient at a point that is not stationary (reading G9). */
typedef struct {
  int *n_accept, *n_reject, *n_feval, *n_newton_unconverged, *status;
  double *h_min, *h_max, *t_end;
  int *n_newton_unconverged_bwd;
  unsigned long long *work;   /* [nenv][6]: work actually done, for the roofline numerator: Newton iterations,
                                 row-iterations (sum over iterations of the rows in the solve) and rows (sum over
                                 evaluations of the rows built) of the forward pass [0..2] and of the reverse sweep [3..5] */
} dmx_stats;

/* Builds the device model.  precision: 64 (double) or 32 (float stage arithmetic; time, step
 * size, error norm, controller and state accumulation stay fp64).  Synchronises the device.
 * Returns 0 and *out on success. */
int dmx_model_create(const dmx_model_desc *desc, int precision, dmx_model **out);
void dmx_model_destroy(dmx_model *m);

/* Sizes derived at create.  np = nbody + 8*npair: parameter vector
 * p = [body_mass(nbody) | pair_friction(npair) | pair_solref(2*npair) | pair_solimp(5*npair)];
 * inertia = mass * inertia_unit.  nc = flattened candidate contacts. */
int dmx_model_np(const dmx_model *m);
int dmx_model_nc(const dmx_model *m);
/* Copies the default parameter vector ([np] doubles) to a HOST buffer. */
int dmx_model_default_params(const dmx_model *m, double *p_host);
/* Lanes per environment the kernels use for this model (1, 8, 16 or 32). */
int dmx_model_lanes(const dmx_model *m);

/* Tape record per accepted step (padded to 16 bytes, written with 16-byte stores): the checkpoint (y_n as nq+nv reals;
 * t_n, h_n as two doubles in both precisions), and - by
 * default - the six stage rates A_1..A_6 (6*nv reals), so that the reverse sweep rebuilds the stage states without
 * re-evaluating F (memory for time, the checkpoint-count knob of PAPER.md:371).  on = 0 keeps the checkpoint only and
 * the reverse sweep recomputes the stages with six F evaluations per step.  Set before sizing / writing a tape. */
int dmx_model_set_tape_stages(dmx_model *m, int on);

/* Checkpoint count knob (PAPER.md:371-375 "memory = number of checkpoints x size of the ODE state", :431 checkpointing
 * trades memory for recomputation).  k = 1 (default): one record per accepted step.  k > 1: the tape keeps a full
 * checkpoint (y_n, t_n, h_n and the first-stage rate) only for the accepted steps 0, k, 2k, ... and, for every step, its signed
 * step size (8 bytes); the reverse sweep re-runs each segment of k steps forward from its checkpoint (same stages, same
 * FSAL rule and step sizes, hence the same states) into a buffer of k full records per resident lane group and sweeps
 * that.  Memory per environment goes from N records to N/k records + 8N bytes (+ k records of scratch per resident
 * group); the sweep costs one extra forward pass.  Gradients equal those of k = 1.  Set before sizing / writing a tape;
 * the call synchronises the device and (re)allocates the segment buffers.  dmx_rollout_*_adjoint and
 * dmx_rollout_backward_noalloc need k = 1. */
int dmx_model_set_checkpoint_stride(dmx_model *m, int k);

/* Bytes of tape for nenv environments with room for tape_steps accepted steps each (uniform slots; no plan). */
size_t dmx_tape_bytes(const dmx_model *m, int nenv, int tape_steps);

/* Launch plan (optional; "the batched loop waits for the slowest environment", PAPER.md:371 memory =
 * checkpoints x state size).  From the accepted-step counts n_accept[nenv] (DEVICE, e.g. the stats of a previous or
 * sizing pass) dmx_tape_plan writes into `plan` (DEVICE buffer of dmx_plan_bytes(nenv)):
 *   - the hand-out order of the work queue: environments by descending n_accept, so the longest chains start first;
 *   - per-environment tape slots of cap(e) = n_accept[e] + n_accept[e]*margin_pct/100 + pad records at the exclusive
 *     prefix sum of the caps, so that the tape holds sum(cap) records instead of nenv * max(cap).
 * The total is dmx_tape_bytes_records(m, nenv, sum_e cap(e)); the caller sizes the tape with the same integer formula.
 * A slot that does not fit the tape buffer, or an environment that outgrows its slot, ends with status 4 (tape full).
 * Pass the same plan to the rollout that writes a tape and to the sweep that reads it.  Enqueues one kernel. */
size_t dmx_plan_bytes(int nenv);
size_t dmx_tape_bytes_records(const dmx_model *m, int nenv, long long total_records);
int dmx_tape_plan(const dmx_model *m, int nenv, const int *n_accept, int margin_pct, int pad, void *plan,
                  size_t plan_bytes, void *cuda_stream);

/* Forward rollout (PAPER.md:41 x_{k+1}=step(x_k,a_k,p); Eq. 5 at PAPER.md:422-425): integrates
 * every environment from t=0 to `horizon` with its own error-controlled step size
 * (PAPER.md:98, 493).
 *   x0      device [nenv, nq+nv] real
 *   ctrl    device [nenv, nknot, nu] real, zero-order hold with knot spacing knot_dt; NULL if nu==0
 *   params  device [nenv, np] real, or NULL for the model defaults
 *   h_replay device [nenv, n_replay] double or NULL: if given, exactly these steps are taken
 *           (a non-positive entry ends the rollout), no error control
 *   xT      device [nenv, nq+nv] real (out)
 *   stats   device arrays (out), may be NULL
 *   tape    device buffer of tape_bytes (16-byte aligned), or NULL for no tape
 *   plan    device buffer written by dmx_tape_plan, or NULL (identity order, uniform tape slots) */
int dmx_rollout(const dmx_model *m, int nenv, const void *x0, const void *ctrl, int nknot, double knot_dt,
                const void *params, double horizon, const dmx_solver_opts *opts, const double *h_replay,
                int n_replay, void *xT, const dmx_stats *stats, void *tape, size_t tape_bytes,
                const void *plan, void *cuda_stream);

/* Forward rollout with tape, then the reverse sweep through the accepted steps with frozen
 * step sizes (discretize-then-optimize).  With cfd_on the vector-Jacobian
 * products are those of the CFD field F~ evaluated on the unmodified trajectory
 * (straight-through estimator, Eq. 4); xT, stats and tape do not depend on
 * cfd_on.
 *   dLdxT     device [nenv, nq+nv] real, ambient gradient of the loss at x_T
 *   dLdx0     device [nenv, 2*nv] real (out), tangent coordinates (translations world frame,
 *             rotations body frame)
 *   dLdctrl   device [nenv, nknot, nu] real (out) or NULL
 *   dLdparams device [nenv, np] real (out) or NULL (skips the parameter directions)
 *   tape      device buffer, required */
int dmx_rollout_grad(const dmx_model *m, int nenv, const void *x0, const void *ctrl, int nknot, double knot_dt,
                     const void *params, double horizon, const dmx_solver_opts *opts, const double *h_replay,
                     int n_replay, const void *dLdxT, int cfd_on, void *xT, void *dLdx0, void *dLdctrl,
                     void *dLdparams, const dmx_stats *stats, void *tape, size_t tape_bytes, const void *plan,
                     void *cuda_stream);

/* Reverse sweep only, over a tape written by dmx_rollout with the same inputs (and the same plan).
 *   stats   NULL, or: stats->status (in, [nenv] or NULL) marks environments to skip (non-zero: zero gradients);
 *           stats->n_newton_unconverged_bwd (out, [nenv] or NULL).  Other fields are ignored. */
int dmx_rollout_backward(const dmx_model *m, int nenv, const void *ctrl, int nknot, const void *params,
                         const dmx_solver_opts *opts, const void *xT, const void *dLdxT, int cfd_on,
                         void *dLdx0, void *dLdctrl, void *dLdparams, const dmx_stats *stats,
                         const void *tape, size_t tape_bytes, const void *plan, void *cuda_stream);

/* The reverse sweep for callers that must not allocate at call time (CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc).  Same arguments, outputs and results as dmx_rollout_backward; the per-lane-group adjoint
 * arrays and the work-queue counter live in a static device array of dmx_noalloc_scratch_bytes() = 16 MiB that every
 * GPU which loads the library holds until the process exits.  The call enqueues two memsets and one kernel and calls no
 * cudaMalloc / cudaFree / allocating library routine.  Limits and rules:
 *   - a model must have been created with the current device current (that is where the array's device address is
 *     taken, once per device); otherwise the call fails;
 *   - the scratch need grows with nenv up to the resident grid (about 4.3 KB per environment for BASELINE config 2, so
 *     ~3800 environments); a larger batch is rejected with an error that states the need and the limit;
 *   - every call on a device shares the array: calls that overlap on the GPU (different streams without ordering
 *     between them) race.  Calls on one stream, or ordered by events, are safe; the array keeps the last call's
 *     contents and each call clears what must start at zero. */
size_t dmx_noalloc_scratch_bytes(void);
int dmx_rollout_backward_noalloc(const dmx_model *m, int nenv, const void *ctrl, int nknot, const void *params,
                                 const dmx_solver_opts *opts, const void *xT, const void *dLdxT, int cfd_on,
                                 void *dLdx0, void *dLdctrl, void *dLdparams, const dmx_stats *stats,
                                 const void *tape, size_t tape_bytes, const void *plan, void *cuda_stream);

/* Optimize-then-discretize (Eq. 6-7; with cfd_on the altered adjoint equations PAPER.md:462-477,
 * Eq. 8-9): the gradient as the solution of the continuous adjoint equations, solved BACKWARDS with its own
 * error-controlled steps under adj_opts (tableau, rtol, atol over the 2*nv adjoint components, controller constants,
 * max_steps = budget of attempted sub-steps per environment; h0 is not used: the first proposal is the last forward
 * step).  Inside an accepted forward step the state is the cubic Hermite interpolant, in the step's chart, of the end
 * values and rates held on the tape (plus one evaluation of F at the end of the step); sub-steps are clipped to the
 * tape's checkpoints.  PAPER.md:452, 473-475 (Fig. 19): with CFD the adjoint equation can be stiff where the forward one
 * is not, and unrolling the (large) forward steps gives wrong gradients whatever the forward tolerance; this call is the
 * remedy.  Same arguments and outputs as dmx_rollout_backward / dmx_rollout_grad, plus
 *   adj_info  device int [nenv, 3] or NULL (out): accepted sub-steps, rejected sub-steps, status (0 ok, 1 sub-step
 *             budget, 2 sub-step underflow, 3 evaluation failed); a failed environment returns zero gradients.
 *   adj_replay device double [nenv, n_adj_replay] or NULL: if given, exactly these sub-steps are taken in order, without
 *             error control (each must end inside or at the end of the current forward step; a non-positive entry or a
 *             sub-step that overshoots fails the environment) - the backward counterpart of h_replay.
 * xT, stats and the tape do not depend on the gradient mode. */
int dmx_rollout_backward_adjoint(const dmx_model *m, int nenv, const void *ctrl, int nknot, const void *params,
                                 const dmx_solver_opts *opts, const dmx_solver_opts *adj_opts, const void *xT,
                                 const void *dLdxT, int cfd_on, void *dLdx0, void *dLdctrl, void *dLdparams,
                                 const dmx_stats *stats, int *adj_info, const double *adj_replay, int n_adj_replay,
                                 const void *tape, size_t tape_bytes, const void *plan, void *cuda_stream);
int dmx_rollout_grad_adjoint(const dmx_model *m, int nenv, const void *x0, const void *ctrl, int nknot, double knot_dt,
                             const void *params, double horizon, const dmx_solver_opts *opts,
                             const dmx_solver_opts *adj_opts, const double *h_replay, int n_replay, const void *dLdxT,
                             int cfd_on, void *xT, void *dLdx0, void *dLdctrl, void *dLdparams, const dmx_stats *stats,
                             int *adj_info, const double *adj_replay, int n_adj_replay, void *tape, size_t tape_bytes,
                             const void *plan, void *cuda_stream);

/* Building blocks exposed for parity tests (one lane-group per state, same device code as the
 * rollouts).  All pointers DEVICE, real typed; n states.
 *   dmx_vector_field: acc[n,nv] = F(q,v,u,p) or F~ when cfd (Eq. 1, 2, 4); nrow[n] rows in the solve.
 *   dmx_vjp_field: (qbar,vbar,ubar,pbar) = kappa^T dF/d(q,v,u,p). */
int dmx_vector_field(const dmx_model *m, int n, const void *x, const void *u, const void *params, int cfd,
                     void *acc, int *nrow, void *cuda_stream);
int dmx_vjp_field(const dmx_model *m, int n, const void *x, const void *u, const void *params, const void *kappa,
                  int cfd, void *qbar, void *vbar, void *ubar, void *pbar, void *cuda_stream);

/* Optimiser step of the paper's applications built on the gradients above (section 5.2: "Adam
 * optimizer with a learning rate of 0.01", "gradient clipping"; PAPER.md:515 E.2: Adam with b1 = 0.5, b2 = 0.9, eps = 1e-6).
 * For every row r of x[nrow][len] with active[r] != 0 (active may be null = all rows):
 *     g_r <- g_r * min(1, clip / ||g_r||_2)      (clip <= 0: no clipping; g itself is not modified)
 *     m <- b1 m + (1 - b1) g_r,   v <- b2 v + (1 - b2) g_r^2
 *     x <- x - lr * (m / (1 - b1^t)) / (sqrt(v / (1 - b2^t)) + eps)          (Kingma & Ba 2015, bias-corrected)
 * t >= 1 is the step counter of this update; mom1 / mom2 are the caller's moment buffers (zero before the first step).
 * x, g, mom1, mom2: DEVICE [nrow][len] of precision 64 / 32 reals; active: DEVICE [nrow] bytes.  Enqueues one kernel
 * on cuda_stream and returns; allocates nothing.  Returns 0, or -1 on bad arguments (dmx_last_error). */
int dmx_adam_step(int precision, int nrow, int len, void *x, const void *g, void *mom1, void *mom2,
                  const unsigned char *active, int t, double lr, double b1, double b2, double eps, double clip,
                  void *cuda_stream);

/* FP64 / FP32 FMA-chain microbenchmark used for the roofline denominator:
 * runs `iters` dependent-chain FMAs x 8 chains per thread on the whole chip and returns the
 * measured FLOP/s (2 per FMA) in *flops_per_s.  Synchronises. */
int dmx_fma_peak(int precision, int iters, double *flops_per_s, double *ms);

/* Diagnostics: per-phase SM-clock counters of the kernels (32 slots, summed over lane groups since the last call);
 * all zero unless the library was compiled with -DDMX_PROF.  Synchronises. */
int dmx_debug_counters(const dmx_model *m, unsigned long long *host32);

const char *dmx_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* DMX_H */
