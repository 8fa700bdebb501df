/*
 * psc.h -- C ABI of the B200-native particle-in-cell hot path of arXiv:1310.7866
 * (Germaschewski et al., "The Plasma Simulation Code").
 *
 * The calls follow the paper's module split (a field pusher with an E method
 * and a B method, a particle pusher, a sort, ghost-point exchange; state in `psc_fields` and
 * `psc_particles`) and the optimised time step of Fig. 8.
 *
 * General rules
 *   - Every pointer is a DEVICE pointer unless its name or comment says "host".
 *   - The library never allocates particle or field storage: the caller owns all buffers (and the
 *     stream) and the library borrows the pointers until the next bind or psc_destroy.  The only
 *     device memory the context owns is a 64-byte status/counter block (and, once psc_marder or
 *     psc_charge_density has been called, one scratch field of the size of E).
 *   - Every call that does device work enqueues it on `stream` (a cudaStream_t passed as void*).
 *     The steady-state calls -- psc_step, psc_push_particles, psc_push_fields, psc_exchange_j,
 *     psc_fill_ghosts, psc_marder_static, psc_patch_loads, psc_particles_gather / _export -- return
 *     without synchronising.  These SYNCHRONISE the stream because they read the device's status
 *     block back: psc_particles_sort (and therefore the first psc_step after a bind, an export or
 *     a psc_step_host, which sorts), psc_status, psc_store_info, psc_profile, psc_step_host.
 *     psc_marder and psc_charge_density cudaMalloc their scratch field on their first call, which
 *     synchronises the whole device once (psc_marder_static never does).
 *   - psc_step / psc_push_particles start with a one-thread gate kernel that may launch the store's
 *     re-layout from the device (tail launches); a stream capture of these calls into a CUDA graph
 *     is therefore not supported by this library version.
 *   - Every call returns 0 (PSC_OK) or a negative PSC_ERR_* code; nothing aborts or throws across
 *     the ABI.  Data-dependent faults are sticky device flags read with psc_status.
 *   - There is no CPU fallback anywhere: without a CUDA device every compute call fails with
 *     PSC_ERR_CUDA.
 *
 * Units and conventions: c = eps0 = mu0 = 1; momentum columns hold
 * u = p/(m_s c); qw = q_s * w; a direction with n[d] == 1 is invariant: no ghosts, no
 * derivative, its coordinate is carried but never advanced.
 *
 * Particle store ("struct of arrays", fp32).  The caller hands over ABSOLUTE
 * positions in [0, n[d]*dx[d]) as n dense entries per column.  Absolute fp32 coordinates have an
 * ulp of up to 6e-5 cells on a 1024-cell axis, which is not enough to keep the deposited current
 * within 1e-5 of the fp64 scheme over several steps, so the first psc_particles_sort moves the
 * particles into the INTERNAL form, the "cell store": positions become in-cell offsets in [0,1)
 * (units of cells), and the particles of cell k (key order of the sort) occupy the slots
 * [base[k], base[k] + count[k]) of the other column set, where base[k] is a multiple of 32 and
 * leaves every cell spare room -- which is why the columns of that set (the `secondary` set of
 * psc_bind_particles) must be psc_particle_capacity(n) entries long, not n.  A push updates particles that stay in their cell in place and hands the
 * others over through per-cell exchange rows in the workspace (see psc_push_particles), so
 * between two pushes some particles live outside the columns.  psc_particles_gather returns a
 * dense copy of everything (offsets + cell keys, or absolute positions) without changing the
 * state; psc_particles_export converts the store back to n dense absolute entries
 * (psc_step_host does so before copying out).  psc_particles_form tells which form is current.
 *
 * Field layout: each of E, B, J is float[3][ez][ey][ex] with ex = n[0] + 2*g (1 if n[0] == 1)
 * etc., x fastest; interior cell i is stored at i + g.  Yee staggering (PAPER.md:141-143,
 * Eq. 20-21):  E[0]=E_x(i+1/2,j,k)  E[1]=E_y(i,j+1/2,k)  E[2]=E_z(i,j,k+1/2);
 * B[0]=B_x(i,j+1/2,k+1/2)  B[1]=B_y(i+1/2,j,k+1/2)  B[2]=B_z(i+1/2,j+1/2,k); J is co-located
 * with E.  Ghost layers hold periodic images.
 */
#ifndef PSC_H
#define PSC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PSC_OK 0
#define PSC_ERR_INVALID_ARG (-1)
#define PSC_ERR_NOT_BOUND (-2)
#define PSC_ERR_NOT_SORTED (-3)
#define PSC_ERR_CFL (-4)
#define PSC_ERR_ALIGN (-5)
#define PSC_ERR_CUDA (-6)
#define PSC_ERR_UNSUPPORTED (-7)
#define PSC_ERR_WORKSPACE (-8)
#define PSC_ERR_SCRATCH_LIMIT (-9) /* psc_marder_static: the grid does not fit the fixed scratch array */

#define PSC_E 0
#define PSC_B 1
#define PSC_J 2

/* sticky device flags (psc_status) */
#define PSC_F_OOB 1u      /* a particle position outside [0, n*dx) was seen by the sort (the particle
                             is filed under the nearest edge cell) */
#define PSC_F_NAN 4u      /* a non-finite momentum was produced; the particle is kept (in its cell, at its
                             last finite offsets), but its current has poisoned J around it */
#define PSC_F_SPECIES 8u  /* a species index outside [0, n_species) was seen by the sort (the
                             particle is treated as species 0) */
#define PSC_F_OVERFLOW 32u /* a particle found no room although the columns / workspace have the
                             sizes psc_particle_capacity / psc_workspace_bytes ask for: lost */
/* (a move of more than one cell, cannot occur: psc_create enforces dt <= dx/2 and
 * |v| < c, so |move| < 1/2 cell; non-finite momenta raise PSC_F_NAN.) */

#define PSC_MAX_SPECIES 8
#define PSC_SCHEME_STANDARD 0
#define PSC_SCHEME_ALTERNATING 1
#define PSC_GHOST 2

typedef struct psc_ctx psc_ctx; /* opaque, host side */

typedef struct {
  int32_t n[3];      /* interior cells x,y,z; n[d] == 1: invariant direction; otherwise >= 4 */
  int32_t ghost;     /* ghost layers in every non-invariant direction; must be PSC_GHOST (2),
                        which suffices for both orders when dt <= min(dx)/2 */
  float dx[3];       /* cell sizes */
  float dt;          /* must satisfy dt <= min over non-invariant d of dx[d]/2 (PSC_ERR_CFL) */
  int32_t order;     /* 1: b1 gather + Villasenor-Buneman; 2: b2 gather + Esirkepov
                         */
  int32_t n_species; /* 1..PSC_MAX_SPECIES */
  const float *q;    /* host array [n_species], charge */
  const float *m;    /* host array [n_species], mass */
  int32_t block[3];  /* sort block ("supercell") in cells; 0: library default;
                        must divide n[d]; 1 along invariant directions */
  int32_t scheme;    /* PSC_SCHEME_STANDARD: every gather weight has the order above;
                        PSC_SCHEME_ALTERNATING: the alternating-order interpolation of PAPER.md:204
                        ("for improved energy conservation"): along a direction in which a field
                        component is half-staggered on the Yee grid its gather weight is one order
                        lower (order 1: b0 instead of b1; order 2: b1 instead of b2); the
                        charge-conserving deposit is unchanged */
} psc_params;

/* One set of particle columns (structure of arrays), each of `capacity`
 * entries (psc_bind_particles).  `id` may be NULL in both sets (then no id is carried).  In a 2-d
 * (yz) run `x`, the coordinate along the invariant direction, may be NULL in both sets (then it
 * is not carried either). */
typedef struct {
  float *x, *y, *z;    /* positions x^{n+1/2}: absolute, or in-cell offsets (internal form) */
  float *ux, *uy, *uz; /* u^n = p/(m c) */
  float *qw;           /* q_s * w */
  int32_t *species;    /* 0 .. n_species-1 */
  int32_t *id;         /* caller's tag, moved with the particle */
} psc_particle_cols;

/* Creates a context.  Validates sizes, block divisibility, the time-step limit.  Host only. */
int psc_create(const psc_params *params, psc_ctx **out);
void psc_destroy(psc_ctx *ctx);

/* Scratch the caller must provide for up to max_particles particles (sort keys, permutation,
 * histograms, scan temporaries, the two exchange buffers of 32 records per cell, the spill
 * list).  Host only. */
size_t psc_workspace_bytes(const psc_ctx *ctx, int64_t max_particles);
/* ws must be 256-byte aligned (PSC_ERR_ALIGN) and at least psc_workspace_bytes large. */
int psc_bind_workspace(psc_ctx *ctx, void *ws, size_t bytes);

/* E, B, J in the layout above.  The caller fills E and B including ghosts, or calls
 * psc_fill_ghosts afterwards.  J need not be initialised. */
int psc_bind_fields(psc_ctx *ctx, float *E, float *B, float *J);
/* Number of floats in one of E/B/J (3 * ex * ey * ez) and the extents; host only. */
int64_t psc_field_elems(const psc_ctx *ctx, int32_t ext[3]);

/* Entries every column of the store set must have for n particles: n + n/8 + 6 sqrt(cells * n) + 56 per
 * cell, rounded up to a multiple of 32 -- every cell of the store gets spare room (an eighth of
 * its population, at least six Poisson standard deviations) and starts on a 128-byte boundary.
 * Host only. */
int64_t psc_particle_capacity(const psc_ctx *ctx, int64_t n);

/* The two column sets have fixed roles.  `primary` is the DENSE set: it holds the n particles the
 * caller hands over (absolute positions, entries [0, n)), receives the n dense entries of
 * psc_particles_export / psc_step_host, and serves as the n-entry scratch of a re-layout; the
 * library never touches an entry beyond n, so its columns need only n entries.  `secondary` is
 * the STORE set: the sort files the particles into it and the pushes update them there; each of
 * its columns has `capacity` >= psc_particle_capacity(n) entries (PSC_ERR_WORKSPACE).  Device
 * memory per particle is therefore (1 + capacity/n) column entries, not 2 * capacity/n.  All
 * columns are 16-byte aligned (PSC_ERR_ALIGN).  Binding marks the particle list as unsorted. */
int psc_bind_particles(psc_ctx *ctx, int64_t n, int64_t capacity, const psc_particle_cols *primary,
                       const psc_particle_cols *secondary);

/* Cell-key counting sort.  key = block-major, cell-minor; stable (ascending
 * input index inside a key).  Afterwards the particles are in the internal form (the cell store
 * above) in sorted order: cell after cell, inside a cell in input order.  Arbitrary input order
 * is accepted.  From absolute columns the keys come from floor(fl32(x * (1/dx))) and the result
 * is written to the store set; from the internal form (sorted,
 * or advanced by psc_push_particles) the input order is the dense order of psc_particles_gather
 * and the keys are the cells the particles are filed under.  psc_sort_result describes this
 * call's permutation.  Synchronises `stream` (it reads the layout statistics back).  psc_step
 * does NOT run this sort in the steady state: see psc_step. */
int psc_particles_sort(psc_ctx *ctx, void *stream);

/* The particle loop of Fig. 8 in one pass over the particles
 * (PAPER.md:603): zero J; per particle gather E,B at x^{n+1/2} (Eq. 11), Boris push
 * p^n -> p^{n+1} (Eq. 27-28), x^{n+1/2} -> x^{n+3/2} (Eq. 26), charge-conserving deposit of
 * j^{n+1}, periodic wrap (on the integer cell index).  Requires the internal
 * form (PSC_ERR_NOT_SORTED otherwise).  In place: a particle that stays in its cell is
 * rewritten where it is (positions and momenta only; q*w, species, id are not touched); a particle
 * that leaves (at most one cell per direction and step) is written as a 32-byte
 * record, tagged with the direction code of its move, into the exchange row of its source cell
 * and is picked up from there by the next psc_push_particles of its destination cell, which
 * files it into a free slot ("reorder on load").  An exchange row holds 32 records
 * and a cell has finite capacity: what does not fit goes to a spill list, and the next
 * psc_push_particles / psc_step first lays the store out again (on the device, no host round
 * trip).  J ghosts are NOT folded on return (psc_exchange_j). */
int psc_push_particles(psc_ctx *ctx, void *stream);

/* FDTD (Eq. 17-18): which == PSC_B: B -= frac*dt*curl+ E;
 * which == PSC_E: E += frac*dt*(curl- B - J) (J interior must be folded).  Interior and ghost
 * points of the updated field are written consistently. */
int psc_push_fields(psc_ctx *ctx, int which, float frac, void *stream);

/* add_and_fill_ghosts_j of Fig. 8 on one GPU: add every ghost value of J onto its periodic
 * image in the interior, then refill the ghosts from the interior. */
int psc_exchange_j(psc_ctx *ctx, void *stream);
/* fill_ghosts of Fig. 7/8 for which in {PSC_E, PSC_B, PSC_J}: ghosts := periodic images. */
int psc_fill_ghosts(psc_ctx *ctx, int which, void *stream);

/* Node charge density ("charge densities on corners"): rho(i,j,k) = sum over all
 * particles of (q w / dV) S(x_p - x_ijk) with the weights of the bound order (b1 / b2, Eq. 31),
 * into the caller's device array float[ez][ey][ex] (the extents of one field component), ghosts
 * = periodic images.  Requires the internal form. */
int psc_charge_density(psc_ctx *ctx, void *stream, float *rho);

/* Marder's correction of Gauss's law (fp32 runs over very many steps drift away
 * from div E = rho; "PSC implements the iterative method by Marder to dissipate violations"):
 * `iters` passes of  E += diffusion * grad+ (div- E - rho)  with rho = psc_charge_density of the
 * current particles (E at the time level of the positions, as stored between two psc_step).
 * `diffusion` is Marder's d * dt (units length^2); a pass multiplies a Fourier mode of the
 * residual by 1 - diffusion * sum_d (2/dx_d)^2 sin^2(k_d dx_d / 2), so it must satisfy
 * diffusion * sum_d 4/dx_d^2 <= 1 (PSC_ERR_CFL).  Requires the internal form.  Uses one scratch
 * field the context allocates on first use (freed by psc_destroy). */
int psc_marder(psc_ctx *ctx, void *stream, float diffusion, int iters);

/* psc_marder for callers that cannot allocate device memory at the point where they apply the
 * correction.  psc_marder cudaMalloc's its scratch field on first use; that is not an option for
 * a time loop that runs while another host thread captures a CUDA graph in the global capture
 * mode (cudaMalloc is forbidden there), for one that cannot take cudaMalloc's implicit
 * device-wide synchronisation, or inside a process whose own pool already holds all of the HBM
 * so that a raw cudaMalloc from a library fails.  This call does the same arithmetic with the same
 * kernels and the same arguments, results and error codes, but keeps rho and the residual in a
 * fixed array that is part of the library's device image, and calls no cudaMalloc, cudaFree or
 * any other allocating routine.
 *   - Limit: the grid including ghosts, ex * ey * ez (psc_field_elems / 3), must not exceed
 *     PSC_MARDER_STATIC_MAX_POINTS (e.g. 64^3 or 1 x 512 x 512 interior cells); a larger grid is
 *     refused with PSC_ERR_SCRATCH_LIMIT before anything is enqueued.  Use psc_marder there.
 *   - Cost: every GPU on which the library is loaded holds the array (3 * 4 *
 *     PSC_MARDER_STATIC_MAX_POINTS bytes = 3.75 MiB) until the process exits.
 *   - The device that owns the bound buffers must be current.  The first call on each device looks
 *     up the array's address on that device (cudaGetSymbolAddress, which may load the module
 *     there); make that first call during set-up, before any stream capture begins.
 *   - The array is shared by every context and every call on a device and keeps the last call's
 *     contents; the call zeroes what must start at zero on `stream`.  Two calls whose device work
 *     can overlap (different streams, different contexts, different host threads) race on it:
 *     order them yourself.  Calls on one stream are ordered by the stream. */
#define PSC_MARDER_STATIC_MAX_POINTS 327680
int psc_marder_static(psc_ctx *ctx, void *stream, float diffusion, int iters);

/* ---- patch-based load balancing (Appendix A) -------------
 * The domain is cut into many more patches than processing elements; the patches are enumerated
 * along a Hilbert-Peano space-filling curve, and the 1-d curve is cut into as many segments as
 * there are ranks so that every rank gets a load matching its capability.  A patch here is
 * patch_blocks[d] sort blocks ("supercells") along direction d (must divide the number of blocks;
 * 1 along an invariant direction), i.e. np[d] = n[d] / (block[d] * patch_blocks[d]) patches. */

/* Load of every patch = its particles + its cells, counted on the device from the
 * cell store (residents by their cell, records waiting in an exchange row by the cell they move
 * to): loads[(pz * np[1] + py) * np[0] + px], a DEVICE array of np[0]*np[1]*np[2] int64.
 * Requires the internal form.  np_out (host, may be NULL) receives np[]. */
int psc_patch_loads(psc_ctx *ctx, void *stream, const int32_t patch_blocks[3], int64_t *loads,
                    int32_t np_out[3]);

/* Hilbert-Peano order of an np[0] x np[1] x np[2] grid of patches (Fig. 5(b)):
 * order[i] (HOST array, np[0]*np[1]*np[2] entries) = row-major index (pz*np[1]+py)*np[0]+px of
 * the i-th patch on the curve.  np[d] == 1 drops that direction (a 2-d curve for a 2-d grid).
 * Extents that are not equal powers of two: the grid is embedded in the enclosing power-of-two
 * cube and the curve's points outside the grid are skipped -- consecutive patches are then no
 * longer always face neighbours (the curve re-enters the grid elsewhere), and the walk costs one
 * visit per point of the cube: a grid whose cube has more than 2^32 points (e.g. 2 x 2 x 65536) is
 * refused with PSC_ERR_UNSUPPORTED.  Host only, no device needed. */
int psc_hilbert_order(const int32_t np[3], int32_t *order);

/* Appendix A: loads[p] (HOST, double, p in CURVE order, n_patches entries, all >= 0),
 * capability[r] (HOST, n_ranks entries, all > 0; e.g. 1 per CPU core and 60 for the
 * rank that drives a GPU) -> count[r] (HOST): rank r takes the next count[r] consecutive patches of
 * the curve.  Every rank gets at least one patch; requires n_patches >= n_ranks >= 1
 * (PSC_ERR_INVALID_ARG).  Host only, no device needed. */
int psc_balance(int64_t n_patches, const double *loads, int32_t n_ranks, const double *capability,
                int32_t *count);

/* The assignment psc_balance's counts stand for: owner[i] (HOST, n_patches entries) = rank of the
 * i-th patch ON THE CURVE (rank 0 takes the first count[0] patches, rank 1 the next count[1], ...).
 * Comparing the owners before and after a re-balance gives the patches that have to move between
 * ranks ("dynamically shifting the assignment of patches"); because the cut points
 * only slide along the curve, a patch moves to a rank whose segment is adjacent on the curve.
 * count[] must be >= 0 and sum to n_patches (PSC_ERR_INVALID_ARG).  Host only. */
int psc_balance_owners(int64_t n_patches, int32_t n_ranks, const int32_t *count, int32_t *owner);

/* One time step, Fig. 8: sort, B half, particle loop, B half,
 * J exchange, E full.  State E^{n+1/2}, B^n, x^{n+1/2}, u^n -> E^{n+3/2}, B^{n+1}, x^{n+3/2},
 * u^{n+1}.  Same fields and the same set of particles (up to the rounding of the atomically
 * summed J) as the calls above in that order.  Only the first step sorts:
 * afterwards the store keeps itself ordered by cell (see psc_push_particles), so a steady-state
 * step reads every particle once and writes its positions and momenta once.  Inside a cell the
 * order is then arbitrary instead of the stable order psc_particles_sort gives. */
int psc_step(psc_ctx *ctx, void *stream);

/* End-to-end form with HOST buffers: copies the host particle columns (n particles) and host
 * E, B (full layout incl. ghosts) into the bound device buffers, runs `nsteps` psc_step, copies
 * particles, E, B, J back, and synchronises the stream.  Host pointers should be pinned.
 * host->id may be NULL iff no id is bound. */
int psc_step_host(psc_ctx *ctx, void *stream, int64_t n, const psc_particle_cols *host,
                  float *hostE, float *hostB, float *hostJ, int nsteps);

/* Inspection of the last psc_particles_sort.  Device pointers into the workspace, valid until
 * the next sort or push:
 * cell_idx[n] (cell of input particle a, natural (k*ny+j)*nx+i; computed on `stream` by this
 * call), perm[n] (sorted position s holds input particle perm[s]), cell_offsets[n_keys+1]
 * (exclusive scan of the key histogram: dense positions, not slots of the store). */
int psc_sort_result(psc_ctx *ctx, void *stream, const int32_t **cell_idx, const int32_t **perm,
                    const int32_t **cell_offsets, int64_t *n_keys);
/* The column set that currently holds the particles: n dense absolute entries
 * (psc_particles_form == 0), or the cell store (== 1: use psc_particles_gather to read it). */
int psc_particles_current(const psc_ctx *ctx, psc_particle_cols *out);
/* 0: absolute positions, 1: internal form (cell store). */
int psc_particles_form(const psc_ctx *ctx);
/* Internal form only: writes a dense copy of all n particles into the caller's device columns
 * `dst` (each >= n entries; x / id may be NULL) without changing any state: cell after cell in
 * key order, a cell's resident particles first, then the records waiting in its exchange row.
 * absolute == 0: positions are in-cell offsets and key[i] (device, >= n entries, may be NULL) is
 * the sort key of the cell they refer to; absolute != 0: x = (cell + offset) * dx, formed in fp64
 * and rounded once.  Entries of a sorted store come out in sorted order. */
int psc_particles_gather(psc_ctx *ctx, void *stream, const psc_particle_cols *dst, int32_t *key,
                         int absolute);
/* Converts the store back to n dense absolute entries (as psc_particles_gather, into the other
 * column set, which becomes the current one).  The list counts as unsorted afterwards.  No-op on
 * absolute columns. */
int psc_particles_export(psc_ctx *ctx, void *stream);
/* Synchronises `stream`; info[0] = largest cell count at the last layout, [1] = slots of the
 * store in use, [2] = re-layouts since psc_create, [3] = particles spilled by the last push,
 * [4] = slots of the per-warp cell image of the particle kernels, [5] = 1 if the last particle
 * push staged its field / J tiles by TMA tensor copies (3-d, order 1, default block, no optional
 * columns), [6] = spilled particles that were filed straight into their cell without a re-layout
 * since psc_create.  Host array. */
int psc_store_info(psc_ctx *ctx, void *stream, int64_t info[8]);
/* Synchronises `stream`, returns and keeps the sticky flags. */
int psc_status(psc_ctx *ctx, void *stream, uint32_t *flags);
/* Kernels and memsets/copies this context has enqueued so far (host counter). */
int64_t psc_launch_count(const psc_ctx *ctx);
/* Last CUDA runtime error code seen by this context (0 if none). */
int psc_last_cuda_error(const psc_ctx *ctx);
/* Per-phase device timing.  After psc_set_option(ctx, "profile", 1) every call brackets its
 * phases with CUDA events recorded on the call's stream (no synchronisation while running; a full
 * event ring is drained with one cudaEventSynchronize).  psc_profile synchronises `stream`, adds
 * the elapsed milliseconds of every completed bracket to ms[PSC_PH_COUNT] and the number of
 * brackets to count[PSC_PH_COUNT] (host arrays), and resets the accumulators.  PSC_PH_SORT spans
 * the whole psc_particles_sort, or inside psc_step the (normally empty) re-layout launches
 * (PSC_PH_SORT_* are its parts); PSC_PH_PUSH is the fused gather-push-deposit kernel launch
 * alone. */
#define PSC_PH_SORT 0
#define PSC_PH_PUSH 1
#define PSC_PH_J_ZERO 2
#define PSC_PH_FIELD_B 3
#define PSC_PH_J_EXCHANGE 4
#define PSC_PH_FIELD_E 5
#define PSC_PH_SORT_COUNT 6
#define PSC_PH_SORT_SCAN 7
#define PSC_PH_SORT_RANK 8
#define PSC_PH_SORT_REORDER 9
#define PSC_PH_MARDER 10
#define PSC_PH_COUNT 16
int psc_profile(psc_ctx *ctx, void *stream, double *ms, int64_t *count);
/* Host-side switches: "profile" (0/1: per-phase event timing), "clear_flags" (reset the sticky
 * device flags).  Unknown names return PSC_ERR_INVALID_ARG. */
int psc_set_option(psc_ctx *ctx, const char *name, int64_t value);
const char *psc_strerror(int code);
const char *psc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PSC_H */
