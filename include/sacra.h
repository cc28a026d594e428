/* sacra.h -- C ABI of libsacra: the B200-native (sm_100a) hot path of SACRA-K's spacetime
 * evolution (arxiv/paper_2607_08743): periodic halo fill, Z4c/BSSN right-hand side with 4th-order
 * finite differences, upwind shift advection and 6th-derivative Kreiss-Oliger dissipation, and the
 * classical RK4 update, on batches of independent uniform FP64 patches; plus the constraint monitor of the same
 * fields (Hamiltonian and momentum constraints and their norms).
 *
 * Citations: PAPER.md:N is a line of the paper's text; "SURVEY 8(c) item k" is the written-out form of
 * the system in SURVEY.md (the paper defers the equations to Hilditch et al. 2013).
 *
 * Conventions common to every call
 *   - All state pointers (u, rhs, u_n, u_in, u_out, acc, work) are DEVICE pointers to FP64 data, 16-byte
 *     aligned, owned by the caller. The library allocates nothing and keeps no pointer after return.
 *   - `p` (npatch patch descriptors) and `prm` are HOST pointers, read during the call only.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream). Every call only
 *     enqueues work on that stream; no call synchronises the device or the stream.
 *   - A "state" is one buffer holding, for every patch, SACRA_NF = 25 fields. Field f of a patch starts at
 *     base + patch_offset + f*field_stride (in doubles) and is a (nz+2ng) x (ny+2ng) x pitch_x array, x
 *     fastest; active cell (i,j,k) is stored at ((k+ng)*(ny+2ng) + (j+ng))*pitch_x + (i+ng).
 *     All states passed to one call share the same layout (the same descriptors address each of them).
 *   - Return value: SACRA_OK (0) or a negative sacra_status. No exceptions cross the ABI; nothing is
 *     written to stdout/stderr. NaN/Inf in the data are not detected.
 *
 * Field order (SURVEY 8 conventions):
 *   0 W | 1-6 gt_xx gt_xy gt_xz gt_yy gt_yz gt_zz | 7 K-hat | 8-13 At_xx..At_zz (same order) |
 *   14-16 Gt^x Gt^y Gt^z | 17 Theta | 18 alpha | 19-21 beta^x..z | 22-24 B^x..z
 */
#ifndef SACRA_H_
#define SACRA_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SACRA_NF 25 /* evolved fields: 1+6+1+6+3+1+1+3+3 */
#define SACRA_NG 3  /* ghost zones per side: reach of the upwind and KO stencils */

typedef enum {
  SACRA_OK = 0,
  SACRA_ERR_NULL = -1,        /* a required pointer is NULL                                        */
  SACRA_ERR_BADARG = -2,      /* n < 6, dx <= 0, non-finite dx/dt, stage outside 1..4, npatch < 1,
                                 pitch/stride/offset too small or negative, forbidden aliasing      */
  SACRA_ERR_UNSUPPORTED = -3, /* ng != 3                                                           */
  SACRA_ERR_ALIGN = -4,       /* pointer not 16-byte aligned, or pitch_x/field_stride/patch_offset
                                 breaks the 16-byte row alignment rule below                       */
  SACRA_ERR_CUDA = -5,        /* a CUDA launch failed (cudaGetLastError)                           */
  SACRA_ERR_TOOLARGE = -6     /* the problem exceeds a fixed capacity of the library
                                 (sacra_constraint_norms_static: SACRA_NORMS_STATIC_MAX_PLANES)    */
} sacra_status;

/* One uniform, cell-centred patch (every box of the hierarchy is such a patch). */
typedef struct {
  int32_t nx, ny, nz;   /* active cells per axis, each >= 6                                          */
  int32_t ng;           /* ghost zones per side; must be 3                                           */
  int64_t pitch_x;      /* doubles per x-row, >= nx + 2*ng, even (rows start 16-byte aligned)        */
  int64_t field_stride; /* doubles between consecutive fields, >= pitch_x*(ny+2ng)*(nz+2ng), even    */
  int64_t patch_offset; /* doubles from a state's base pointer to field 0 of this patch, >= 0;
                           (patch_offset + ng) must be even, so that active cell i=0 of every row is
                           16-byte aligned                                                           */
  double dx;            /* grid spacing, dx = dy = dz > 0                                            */
  double dt;            /* full RK4 step of this patch (Courant factor times dx)        */
} sacra_patch_t;

/* Parameters of the evolution system. */
typedef struct {
  double kappa1, kappa2;   /* Z4c constraint damping                    */
  double eta;              /* Gamma-driver damping, Eq. 8                             */
  double shift_coef;       /* coefficient of B^i in Eq. 7: 0.75                       */
  double ko_sigma;         /* Kreiss-Oliger strength; Q = sigma h^5/64 (D+D-)^3       */
  int32_t lapse_uses_khat; /* Eq. 6 source: 1 -> -2 alpha K-hat (default reading),
                              0 -> -2 alpha (K-hat + 2 Theta)                                       */
  int32_t flags;           /* 0, or SACRA_FLAG_* values or'ed together                               */
} sacra_params_t;

/* sacra_params_t.flags */
#define SACRA_FLAG_SKIP_INCREMENT 1 /* stage 4 of the RK4 step does not store the increment S to acc (SURVEY 8(c)
                                       item 11: "this write may be skipped outside verification"): one field pass
                                       less per step; the contents of acc are then unspecified after stage 4 / after
                                       sacra_rk4_step. u_out is the same bit for bit.                             */

/* Periodic halo fill (stands in for the paper's ghost exchange).
 * For every field of every patch, each storage cell with an index outside the active range takes the
 * value of the active cell with per-axis wrapped index; faces, edges and corners. In place on u. Pitch
 * padding beyond nx+2ng is not touched. */
int sacra_fill_ghosts(const sacra_patch_t* p, int npatch, double* u, void* cuda_stream);

/* Halo fill with a boundary mode per axis (axis_mode: HOST int32_t[3], x y z), SURVEY 8(f) f-2:
 *   SACRA_BC_PERIODIC  as sacra_fill_ghosts;
 *   SACRA_BC_MIRROR    reflection symmetry about both faces of the axis (PAPER.md:125 imposes it at z = 0): the ghost
 *                      cell m+1 cells outside a face takes the active cell m cells inside it, times the parity of the
 *                      field under x^a -> -x^a: -1 for Gt^a, beta^a, B^a and for the gt / At components with exactly
 *                      one index a, +1 otherwise; cells reflected along several axes take the product.
 * In place on u; all patches of the call use the same modes. */
#define SACRA_BC_PERIODIC 0
#define SACRA_BC_MIRROR 1
int sacra_fill_ghosts_bc(const sacra_patch_t* p, int npatch, const int32_t* axis_mode, double* u, void* cuda_stream);

/* Physical boundaries per patch and face (section 2.2.2).
 * face[] order: x- x+ y- y+ z- z+. Modes: SACRA_BC_PERIODIC and SACRA_BC_MIRROR as above (PERIODIC on both faces of an
 * axis or on neither); SACRA_BC_SOMMERFELD: outer boundary with the outgoing-wave condition Eq. 13;
 * SACRA_BC_NONE: the ghost cells behind the face belong to somebody else (e.g. sacra_prolong_ghosts) and are left alone.
 * origin: coordinates of the centre of active cell (0,0,0); active cell (i,j,k) sits at origin + (i,j,k) dx (Eq. 13
 * needs x^i / r; the origin of the coordinates must not be a cell of a Sommerfeld boundary shell: every call that
 * evaluates Eq. 13 returns SACRA_ERR_BADARG, before launching anything, if such a cell has r = 0).
 * Reading of Eq. 13 (the paper gives no discretisation): on the BOUNDARY SHELL -- the active cells
 * within 3 cells of a SOMMERFELD face -- the right-hand side of all 25 fields is
 *     d_t Q = -( x^i d_i Q + Q ) / r,   Q = field - flat value (1 for W, gt_xx, gt_yy, gt_zz, alpha; 0 otherwise),
 * with 4th-order differences that use existing cells only: centred (-1 8 0 -8 1)/12h where it fits, else the lopsided
 * (-3 -10 18 -6 1)/12h, else the one-sided (-25 48 -36 16 -3)/12h stencil pointing inwards; no KO term. Everywhere else
 * the Z4c right-hand side applies (its stencils reach 3 cells, so it never reads a ghost cell behind a SOMMERFELD face;
 * those ghost cells are neither read for a kept result nor written). */
#define SACRA_BC_SOMMERFELD 2
#define SACRA_BC_NONE 3
typedef struct {
  double origin[3];
  int32_t face[6];
} sacra_boundary_t;

/* Halo fill with a mode per patch and face (bnd: HOST array of npatch entries). A ghost cell takes the active cell
 * obtained by wrapping / reflecting every axis along which it lies outside; if one of those faces is SOMMERFELD or
 * NONE the cell is left alone. */
int sacra_fill_ghosts_faces(const sacra_patch_t* p, int npatch, const sacra_boundary_t* bnd, double* u, void* cuda_stream);

/* Eq. 13 on the boundary shells: rhs receives the 25 Sommerfeld right-hand sides on the shell cells of every patch;
 * all other cells of rhs are not touched. u: ghosts behind non-SOMMERFELD faces filled. rhs must not overlap u. */
int sacra_sommerfeld_rhs(const sacra_patch_t* p, int npatch, const sacra_boundary_t* bnd, const double* u, double* rhs,
                         void* cuda_stream);

/* sacra_rk4_substep / sacra_rk4_step with physical boundaries: k is the Z4c right-hand side outside the boundary shells
 * and Eq. 13 inside them (two kernels per substage: the fused substage kernel skips the shell cells, a small kernel
 * applies the same stage table there); the halo fills of the step use the face modes. Same argument rules. */
int sacra_rk4_substep_bc(const sacra_patch_t* p, int npatch, const sacra_params_t* prm, const sacra_boundary_t* bnd,
                         int stage, const double* u_n, const double* u_in, double* u_out, double* acc, void* cuda_stream);
int sacra_rk4_step_bc(const sacra_patch_t* p, int npatch, const sacra_params_t* prm, const sacra_boundary_t* bnd, double* u,
                      double* work, int64_t state_doubles, void* cuda_stream);

/* Z4c right-hand side including KO dissipation, F(u) (PAPER.md:49-73,
 * PAPER.md:99). u: ghosts already filled (read only). rhs: the 25 RHS values are written on active cells;
 * ghost cells and padding of rhs are not touched. rhs must not alias u. */
int sacra_z4c_rhs(const sacra_patch_t* p, int npatch, const sacra_params_t* prm, const double* u,
                  double* rhs, void* cuda_stream);

/* One classical RK4 substage. With k = F(u_in) on active cells:
 *   stage 1: u_out = u_n + (dt/2) k ; acc  = k          (requires u_in = u_n)
 *   stage 2: u_out = u_n + (dt/2) k ; acc += 2k
 *   stage 3: u_out = u_n + dt k     ; acc += 2k
 *   stage 4: S = (acc + k) * (1/6)  ; u_out = u_n + dt S ; acc = S
 * u_in: ghosts filled (read through the stencil). u_n: read at active cells only. u_out, acc: active
 * cells written, ghosts not touched. u_out must not alias u_in; u_out may alias u_n (centre-only access);
 * acc must alias none of the others. At stage 1 acc is write-only.
 * Aliasing is checked on whole states: any two of the four buffers must either be the same pointer, where the table
 * allows it (u_n = u_in, required at stage 1; u_out = u_n), or disjoint address ranges of the extent the patch
 * descriptors span -- a partial overlap returns SACRA_ERR_BADARG, like every other forbidden aliasing. */
int sacra_rk4_substep(const sacra_patch_t* p, int npatch, const sacra_params_t* prm, int stage,
                      const double* u_n, const double* u_in, double* u_out, double* acc,
                      void* cuda_stream);

/* One full RK4 step: for s = 1..4 { fill_ghosts(stage input); rk4_substep(s) }; fill_ghosts(result).
 * u: in = state n (ghosts need not be filled), out = state n+1 with ghosts filled.
 * work: 3 states back to back, each `state_doubles` long (two stage buffers and acc). On return
 * work + 2*state_doubles holds S, the increment per unit dt, on active cells (unless prm->flags has
 * SACRA_FLAG_SKIP_INCREMENT). Bitwise identical to the nine-call sequence above. u must not overlap
 * [work, work + 3*state_doubles). Every call of the library only enqueues kernels on cuda_stream, so a step can be
 * captured into a CUDA graph by the caller (the tiny configurations are launch-bound: bench.py --all-configs). */
int sacra_rk4_step(const sacra_patch_t* p, int npatch, const sacra_params_t* prm, double* u,
                   double* work, int64_t state_doubles, void* cuda_stream);

/* Constraint monitor (Eqs. 20-21, vacuum): Hamiltonian constraint H = R + K^2 - K_ij K^ij and
 * momentum constraint M^i = D_j (K^ij - gamma^ij K) of the physical metric gamma_ij = gt_ij / W^2 with
 * K_ij = (At_ij + gt_ij K / 3) / W^2, K = K-hat + 2 Theta; 4th-order centred differences.
 * u: ghosts already filled (read only). con: a state-shaped DEVICE buffer (same descriptors as u); fields 0..3 of
 * every patch receive H, M^x, M^y, M^z on active cells; ghosts, padding and fields 4..24 are not touched.
 * con must not alias u. */
int sacra_constraints(const sacra_patch_t* p, int npatch, const double* u, double* con, void* cuda_stream);

/* Volume-normalised L2 norms of the four constraints over the active cells of all patches (Eq. 22):
 * norms[c] = sqrt( sum_cells C_c^2 dV / sum_cells dV ), dV = dx^3 of the cell's patch.
 * con: output of sacra_constraints. scratch: DEVICE buffer of at least sacra_constraint_scratch_doubles(p, npatch)
 * doubles (4 per active z-plane). norms: DEVICE double[4], written when the stream reaches the call.
 * The reduction order is fixed: the same input gives the same bits on every run. */
int sacra_constraint_norms(const sacra_patch_t* p, int npatch, const double* con, double* scratch, double* norms,
                           void* cuda_stream);
int64_t sacra_constraint_scratch_doubles(const sacra_patch_t* p, int npatch);

/* The same norms for callers that have no device memory left to give and may not ask the CUDA runtime for more.
 * Who that is: an evolution code sizes its state buffers to fill the GPU at start-up and hands everything to its own
 * arena; the monitor is then called from inside the time loop every step, where a cudaMalloc is not
 * an option - it synchronises the whole device, which stalls the streams that overlap the halo exchange with the
 * substage kernels - and where there may simply be nothing left to allocate. sacra_constraint_norms asks such a
 * caller for a scratch buffer; this call does not.
 *
 * Same arguments as sacra_constraint_norms without `scratch`, same kernels, same reduction order, hence the same bits
 * in `norms`. The per-plane partial sums go to an array that lives inside the library image: 4 x
 * SACRA_NORMS_STATIC_MAX_PLANES doubles = 128 KiB of device memory, held by every GPU that loads libsacra from
 * the moment it loads it until the process exits, whether this call is used or not.
 *
 *   - Limit: the active z-planes of all patches together (sum of nz) must not exceed
 *     SACRA_NORMS_STATIC_MAX_PLANES; otherwise SACRA_ERR_TOOLARGE is returned and nothing is launched. (256^3 has
 *     256 planes, the 8 x 64^3 batch 512.) Larger batches: sacra_constraint_norms with the caller's buffer.
 *   - The call itself calls no cudaMalloc / cudaFree and no library routine that allocates.
 *   - First call on each device: with that device current, the library looks the array's device address up
 *     (cudaGetSymbolAddress, return code checked -> SACRA_ERR_CUDA) and keeps it; later calls on that device reuse
 *     it. Make this first call during set-up, outside any stream capture.
 *   - All calls on one device share the one array, and it keeps what the last call left in it. Nothing in it has to
 *     start at zero: each call overwrites every entry it later reads, so stale contents are harmless and nothing is
 *     cleared. Two calls whose kernels can run at the same time on the same device (different streams, no
 *     dependency between them) race on the array and give garbage in both `norms`; order them on one stream or with
 *     an event. */
#define SACRA_NORMS_STATIC_MAX_PLANES 4096
int sacra_constraint_norms_static(const sacra_patch_t* p, int npatch, const double* con, double* norms,
                                  void* cuda_stream);

/* Spatial inter-level operators of the box-in-box hierarchy, 2:1 refinement on
 * cell-centred staggered grids. `parent` and `child` are ONE patch each (HOST pointers; the child has half the
 * spacing and even nx, ny, nz); org: HOST int32_t[3], the parent ACTIVE-cell index of the coarse cell that holds the
 * child's active cells 0 and 1 along each axis (its centre lies midway between them). All 25 fields.
 *   sacra_restrict        every parent cell org + m, 0 <= m < n_child / 2 per axis, is overwritten with the 4-point
 *                         per axis Lagrange interpolant of the child data at its centre (weights -1 9 9 -1 / 16 on child
 *                         cells 2m-1 .. 2m+2; the child's ghost cells are read at the patch edges and must be valid).
 *                         The covered cells must be active cells of the parent.
 *   sacra_prolong_ghosts  every ghost cell of the child (faces, edges, corners) is overwritten with the 6-point per
 *                         axis Lagrange interpolant of the parent data at its centre (a quarter of a parent spacing
 *                         off the parent cell that holds it). Parent cells org + floor(i/2) - 3 .. + 3 are read for
 *                         child cells i = -3 .. n+2: they must lie in the parent's storage (ghosts included, valid).
 * The child's spacing must be half the parent's; the two states must not overlap. */
int sacra_restrict(const sacra_patch_t* parent, const sacra_patch_t* child, const int32_t* org, double* u_parent,
                   const double* u_child, void* cuda_stream);
int sacra_prolong_ghosts(const sacra_patch_t* parent, const sacra_patch_t* child, const int32_t* org,
                         const double* u_parent, double* u_child, void* cuda_stream);

/* Time interpolation of the refinement-boundary data and the Berger-Oliger step of a parent / child pair (SURVEY 8(f)
 * f-3; the child advances with a halved time step, two steps per parent step; its boundary data at the
 * substeps "are interpolated between the parent time levels, at first order in the very first time step of a run and at
 * second order thereafter"). theta = (t - t_n) / dt_parent.
 *   sacra_time_weights   HOST function, no GPU work: weights of the parent time levels at theta. nlevels = 2: the line
 *                        through U^n, U^n+1 (w[2] = 0); nlevels = 3: the parabola through U^n-1, U^n, U^n+1. w: HOST double[3].
 *   sacra_lincomb        out = (w[0] u0 + w[1] u1) [+ w[2] u2] on every storage cell (ghosts included) of ONE patch, all
 *                        25 fields; w: HOST double[3]; out must not overlap the inputs.
 *   sacra_subcycle_step  one step of the pair: (1) the parent takes one RK4 step with its boundary modes
 *                        (sacra_rk4_step_bc); (2) the child takes two RK4 steps of dt/2: before every substage the ghost
 *                        cells of the stage input are prolonged (sacra_prolong_ghosts) from the parent levels
 *                        interpolated to the substage time theta = (m + c_s)/2, m = 0, 1, c = (0, 1/2, 1/2, 1); (3) the
 *                        child's ghosts are prolonged from the new parent state, the child is restricted onto the
 *                        covered parent cells (sacra_restrict) and the parent's ghosts are refilled.
 *                        u_parent_prev: on entry U^n-1 if have_prev != 0 (else ignored), on return U^n (the state the
 *                        step started from). work_parent: 5 x parent_doubles, work_child: 3 x child_doubles doubles.
 *                        child->dt must be parent->dt / 2; geometry rules as for sacra_prolong_ghosts. */
int sacra_time_weights(int nlevels, double theta, double* w);
int sacra_lincomb(const sacra_patch_t* p, int nlevels, const double* u0, const double* u1, const double* u2, const double* w,
                  double* out, void* cuda_stream);
int sacra_subcycle_step(const sacra_patch_t* parent, const sacra_patch_t* child, const int32_t* org,
                        const sacra_params_t* prm, const sacra_boundary_t* parent_bnd, double* u_parent,
                        double* u_parent_prev, int have_prev, double* u_child, double* work_parent,
                        int64_t parent_doubles, double* work_child, int64_t child_doubles, void* cuda_stream);

/* A hierarchy of nested levels ("fixed levels, each a single cubic patch"): level l + 1 is the child of
 * level l (half its spacing, half its time step, nested at parent index org). One call advances level 0 by one step and
 * every finer level by its two, four, ... steps, recursively: the pair step above applied at every level -- a level takes
 * its RK4 step (level 0 with its boundary modes; level l > 0 with the ghosts of every substage input prolonged from its
 * parent's time levels U^n-1, U^n, U^n+1 at the substage time, first order while the parent has no U^n-1 yet), then its
 * child takes two steps, the child is restricted onto it and its own ghosts are refilled (level 0: boundary modes;
 * l > 0: from the parent at the time just reached). With two levels this is sacra_subcycle_step, bit for bit.
 * levels: HOST array of nlevels entries (<= 16), updated (nsteps). All pointers inside are as described per field. */
typedef struct {
  const sacra_patch_t* patch; /* HOST: the level's patch                                                            */
  int32_t org[3];             /* position in the parent, as for sacra_prolong_ghosts (level 0: ignored)             */
  int32_t pad_;               /* set to 0                                                                           */
  double* u;                  /* DEVICE: the level's state (ghosts valid on entry and on return)                    */
  double* u_prev;             /* DEVICE: U^n-1 of the level; written by every step, read when nsteps > 0            */
  double* work;               /* DEVICE: 5 x state_doubles                                                          */
  int64_t state_doubles;
  int64_t nsteps;             /* steps the level has taken so far (0 at the start of a run); updated by the call    */
} sacra_level_t;
int sacra_hierarchy_step(sacra_level_t* levels, int nlevels, const sacra_params_t* prm, const sacra_boundary_t* bnd0,
                         void* cuda_stream);

/* Halo exchange between the patches of a block decomposition over several GPUs (the
 * 3 ghost layers of every field at every face are packed into a buffer and exchanged with the neighbouring rank before
 * each RK substage). ONE patch per call. axis 0, 1, 2 = x, y, z; side 0 = low face, 1 = high face.
 *   sacra_face_doubles   doubles in a face buffer of the axis: 25 fields x 3 layers x the whole STORAGE extent of the two
 *                        other axes (their ghost cells travel too: exchanging x, then y, then z fills edges and corners).
 *   sacra_pack_face      buf <- the 3 outermost ACTIVE layers at the face, layout [field][layer][slower][faster] (layer
 *                        and the two other axes in increasing storage index).
 *   sacra_unpack_face    the 3 GHOST layers behind the face <- buf (same layout). The buffer a rank packs at its high
 *                        face is what its high neighbour unpacks at its low face, and vice versa.
 * The transfer itself is the caller's (paper_2607_08743_b200/halo.py: torch.distributed point-to-point over NCCL). */
int64_t sacra_face_doubles(const sacra_patch_t* p, int axis);
/* Overlap of the exchange with the computation (PAPER.md:378 lists it as future work): sacra_rk4_substep in two parts.
 * exchange_faces: HOST int32_t[6] (x- x+ y- y+ z- z+), non-zero where the ghosts behind the face come from an exchange.
 *   SACRA_PART_INTERIOR  the active cells more than 3 cells away from every flagged face: they read no exchanged ghost
 *                        cell, so this part can run while the messages are in flight;
 *   SACRA_PART_SHELL     the other active cells, after the unpack (tiles without such a cell are skipped).
 * The two parts write disjoint cells; together they give sacra_rk4_substep bit for bit. Same argument rules. */
#define SACRA_PART_INTERIOR 1
#define SACRA_PART_SHELL 2
int sacra_rk4_substep_part(const sacra_patch_t* p, int npatch, const sacra_params_t* prm, int stage, int part,
                           const int32_t* exchange_faces, const double* u_n, const double* u_in, double* u_out, double* acc,
                           void* cuda_stream);
int sacra_pack_face(const sacra_patch_t* p, const double* u, int axis, int side, double* buf, void* cuda_stream);
int sacra_unpack_face(const sacra_patch_t* p, double* u, int axis, int side, const double* buf, void* cuda_stream);

/* Static description of a status code (never NULL). */
const char* sacra_strerror(int code);

/* Library version, "major.minor" */
const char* sacra_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SACRA_H_ */
