/*
 * vg.h -- C ABI of libvg: batched solid-geometry navigation queries on one NVIDIA B200 (sm_100a).
 *
 * The operations are the three questions the paper asks of the geometry for every particle
 * (sec. III.C):
 *     "Is the particle inside or outside the solid?"                                   -> vg_inside
 *     "What is the minimal distance between the particle and the border of the solid?" -> vg_safety_to_in/out
 *     "What is the maximal step length for a particle with a given velocity and
 *      direction?"                                                                     -> vg_distance_to_in/out
 * and the navigation step that uses them (the distance to the geometric border
 * competes with the physics step; "coordinate transformations and distance calculations")
 *                                                                                      -> vg_compute_step.
 * The paper defines no solid and no formula; the exact meaning of every query is the reading
 * R1-R21 of SURVEY.md sec. 8(c), restated in DESIGN.md sec. 3 together with R22-R32 (the tree of volumes
 * vg_world_*, polycone z steps, boolean solids and CSG trees vg_boolean_create, start points on a surface).
 * In one line each:
 *   Inside        VG_INSIDE if sdf(p) < -kTol, VG_OUTSIDE if sdf(p) > +kTol, else VG_SURFACE (kTol = 1e-9)
 *   SafetyToIn    +sdf(p), SafetyToOut  -sdf(p): exact signed Euclidean distance to the surface (for a
 *                 boolean: the composed bound of R29, which never over-estimates it)
 *   DistanceToIn  -1 if p is inside; else the first t > 0 with p + t d on the surface; +inf if none or > step_max
 *   DistanceToOut -1 if p is outside; else likewise
 *   ... from a start point of class VG_SURFACE (R32; a particle "transported to the border" starts its
 *                 next step there): the ray starts ON the crossing it sits on -- moving inward DistanceToIn = 0 and
 *                 DistanceToOut = the chord to the exit; moving outward DistanceToOut = 0 and DistanceToIn = the
 *                 next entry (+inf for a convex solid).  Every distance returned is -1, >= 0 or +inf.  The kernels
 *                 count a crossing of the wanted sense as lying at the start when its ray parameter is > -5e-7
 *                 (VG_KRAYTOL) and clamp at 0: exact for a band point unless the ray grazes the surface it sits on
 *                 at |n.d| < 2e-3 or another surface lies within 1e-6.
 *   ComputeStep   lexicographic min of (distance, index) over the mother's DistanceToOut (index -1) and every
 *                 daughter's DistanceToIn in its local frame p_i = R_i p + b_i, d_i = R_i d; (step_max, -2)
 *                 if the physics step step_max is shorter.
 *
 * Conventions for every entry point
 *   - Track arrays x, y, z, dx, dy, dz and every output array are DEVICE pointers owned by the caller,
 *     n elements each, FP64 struct-of-arrays (six separate arrays), 8-byte aligned.  When all of them
 *     are 16-byte aligned the 128-bit vectorised path is taken; otherwise a 64-bit path (never an
 *     error, never a host fallback).  Outputs must not alias inputs.
 *   - Shape parameters and placement matrices are HOST pointers, read during the create call only.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Calls enqueue
 *     work and return; they never synchronise.  The caller keeps the arrays alive until the stream
 *     has passed the call.
 *   - Directions must be unit vectors to rounding (not checked, not renormalised).
 *   - Return value: VG_OK or a negative vg_status; vg_last_error() gives a thread-local message.
 *     n == 0 is VG_OK and launches nothing.  No exceptions, no abort, no output to stdout/stderr.
 *   - Handles are immutable after create and may be used concurrently from several host threads
 *     and streams.  A handle belongs to the CUDA device that was current when it was created.
 *   - There is no CPU implementation behind this interface: without a CUDA device every compute
 *     call returns VG_ERR_CUDA.
 */
#ifndef VG_H
#define VG_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct vg_shape vg_shape;   /* opaque solid; owned by the library until vg_shape_destroy          */
typedef struct vg_volume vg_volume; /* opaque mother + placed daughters; does NOT own the vg_shape objects */

typedef enum { VG_BOX = 0, VG_ORB = 1, VG_TUBE = 2, VG_CONE = 3, VG_TRD = 4, VG_POLYCONE = 5,
               VG_BOOLEAN = 6 /* made by vg_boolean_create only */ } vg_kind;

enum { VG_OUTSIDE = 0, VG_SURFACE = 1, VG_INSIDE = 2 }; /* values written by vg_inside */

typedef enum {
    VG_OK = 0,
    VG_ERR_ARG = -1,   /* null pointer, negative n, misaligned (not 8-byte) array, bad step_max      */
    VG_ERR_PARAM = -2, /* shape / volume parameters rejected by validation                           */
    VG_ERR_ALIGN = -3, /* reserved                                                                   */
    VG_ERR_CUDA = -4,  /* CUDA runtime error (no device, launch failure); message has the CUDA text  */
    VG_ERR_NOMEM = -5  /* host or device allocation failed                                           */
} vg_status;

#define VG_KTOLERANCE 1e-9   /* BASELINE.json: kTolerance; half-width of the surface band (R6)        */
#define VG_KRAYTOL 5e-7      /* R32: a crossing this little behind the start point lies AT it         */
#define VG_MAX_ZPLANES 32    /* polycone                                                              */
#define VG_MAX_DAUGHTERS 256 /* per volume                                                            */
#define VG_HIT_MOTHER (-1)   /* vg_compute_step: the mother's boundary limits the step                */
#define VG_HIT_STEPMAX (-2)  /* vg_compute_step: step_max (the physics step) limits it   */

/*
 * vg_shape_create -- build a solid (solids as closed point sets, sec. 8(c) c.1).
 * `params` (HOST, nparams doubles, lengths unitless, angles in radians):
 *   VG_BOX      [hx, hy, hz]                               half-lengths, |x|<=hx, |y|<=hy, |z|<=hz
 *   VG_ORB      [r]                                        x^2+y^2+z^2 <= r^2
 *   VG_TUBE     [rmin, rmax, dz, sphi, dphi]               |z|<=dz, rmin<=rho<=rmax, phi in [sphi, sphi+dphi]
 *   VG_CONE     [rmin1, rmax1, rmin2, rmax2, dz, sphi, dphi]  radii linear in z, index 1 at z=-dz, 2 at z=+dz
 *   VG_TRD      [dx1, dx2, dy1, dy2, dz]                   half-lengths, index 1 at z=-dz, 2 at z=+dz
 *   VG_POLYCONE [sphi, dphi, nz, z_0, rmin_0, rmax_0, ..., z_{nz-1}, rmin_{nz-1}, rmax_{nz-1}]
 *               radii linear between consecutive z-planes, z non-decreasing, 2 <= nz <= VG_MAX_ZPLANES.  Two planes
 *               at the same z are a STEP (reading R26): the radii jump there and the solid gets an
 *               annular face at that z.  A step may not sit at the first or last plane, at most two planes share a z,
 *               and the radial ranges on the two sides of a step must overlap.
 *   dphi >= 2 pi (as FP64) means the full revolution.
 * Validation (VG_ERR_PARAM): wrong nparams, non-finite values, lengths <= 0, rmin < 0, rmin >= rmax at any
 * plane, dphi <= 0, nz out of range or not an integer, z decreasing, a z step that breaks the rules above.
 * On success *out receives a handle; derived constants are computed once here on the host.  For a polycone
 * the candidate grid of its safeties (DESIGN.md sec. 6.2, 65 KiB; 193 KiB with a phi cut) is built here and placed on the CURRENT device if
 * there is one; on another device, or without one at create time, the safeties run the ordered-walk kernel instead.
 */
int vg_shape_create(vg_kind kind, const double *params, int nparams, vg_shape **out);

/*
 * vg_boolean_create -- the boolean solid C = A op B of two primitives ("boolean operations", PAPER.md:110
 * "logical operations"; readings R27-R29 in DESIGN.md).  A sits in the frame of C; `xform_b` (HOST,
 * 12 doubles, row-major 3x4 [R | b], orthonormal R) maps the frame of C to the frame of B.  A and B: box, orb, tube,
 * cone, trd, or a boolean made by this call (reading R31: a CSG tree; at most 8 primitives per tree, VG_ERR_PARAM
 * beyond); their constants are copied.  Two primitives run kernels specialised per pair of kinds, a tree is flattened
 * into a program over its primitives and runs the general kernel (vg_csg.cu).  A or B may also be a POLYCONE when the
 * other one is a primitive or a polycone: its constants are placed in memory of the CURRENT device (VG_ERR_CUDA
 * without one; queries must run on that device) and the general two-operand kernel answers (vg_boolx.cu); such a
 * boolean is not an operand of another boolean (VG_ERR_ARG), but it is a placed solid like any other: a node of a
 * world, the mother or a daughter of a volume (the world / volume copies the polycones' constants once more).
 * The result is a vg_shape of kind VG_BOOLEAN that every query below accepts ("operand" read recursively for a tree):
 *   Inside       combines the operands' classes: union INSIDE if either is, OUTSIDE if both are; intersection INSIDE if
 *                both are, OUTSIDE if either is; subtraction (A minus B) INSIDE if A INSIDE and B OUTSIDE, OUTSIDE if A
 *                OUTSIDE or B INSIDE; SURFACE otherwise (R27);
 *   distances    the first t > 0 at which the membership of C along the ray flips, +inf if none, -1 on the wrong side
 *                (R28; the operands' memberships follow from their crossings along the whole line, so a start point on
 *                an operand's surface that is hidden inside the other operand is an ordinary inside point of C); R32
 *                from a start point of class SURFACE; a ray that clips an operand through a chord shorter than
 *                VG_KRAYTOL passes that operand's two crossings like any others (it is never held there);
 *   safeties     the composed bound sdf_C = min(sdfA, sdfB) / max(sdfA, sdfB) / max(sdfA, -sdfB): it has the sign of the
 *                membership and never over-estimates the distance to the surface of C, but unlike the primitives'
 *                safeties it is not the exact distance everywhere (R29).
 * A boolean (of two primitives or a tree) can be a node of a world and the mother or a daughter of a volume.
 */
typedef enum { VG_UNION = 0, VG_INTERSECTION = 1, VG_SUBTRACTION = 2 } vg_bool_op;
int vg_boolean_create(int op, const vg_shape *a, const vg_shape *b, const double *xform_b, vg_shape **out);
void vg_shape_destroy(vg_shape *shape); /* NULL is allowed */
int vg_shape_kind(const vg_shape *shape); /* the vg_kind, or VG_ERR_ARG for NULL */

/* Inside classification of n points.  cls: DEVICE int32[n]. */
int vg_inside(const vg_shape *shape, const double *x, const double *y, const double *z, int64_t n, int32_t *cls,
              void *stream);

/* DistanceToIn / DistanceToOut of n tracks.
 * step_max >= 0, may be +inf; a crossing farther than step_max is reported as +inf.  dist: DEVICE double[n]. */
int vg_distance_to_in(const vg_shape *shape, const double *x, const double *y, const double *z, const double *dx,
                      const double *dy, const double *dz, double step_max, int64_t n, double *dist, void *stream);
int vg_distance_to_out(const vg_shape *shape, const double *x, const double *y, const double *z, const double *dx,
                       const double *dy, const double *dz, double step_max, int64_t n, double *dist, void *stream);

/* SafetyToIn = +sdf, SafetyToOut = -sdf of n points (exact, signed).
 * safety: DEVICE double[n]. */
int vg_safety_to_in(const vg_shape *shape, const double *x, const double *y, const double *z, int64_t n,
                    double *safety, void *stream);
int vg_safety_to_out(const vg_shape *shape, const double *x, const double *y, const double *z, int64_t n,
                     double *safety, void *stream);

/*
 * vg_query_all -- the five answers of n tracks in one call (a basket of particles in one volume asks all three
 * questions of PAPER.md:110-114 every step).  Same results, element by element, as the five
 * calls above.  Any output pointer may be NULL (that answer is skipped; at least one must be given).  When all five
 * are given and the solid is not a boolean (for a polycone: and every array is 16-byte aligned), ONE fused kernel reads the six track arrays once (48 B per track
 * instead of 168 B) and writes the five results; otherwise the call enqueues one kernel per requested answer.
 * cls: DEVICE int32[n]; the other four: DEVICE double[n]; dx, dy, dz and step_max as for vg_distance_to_in.
 */
int vg_query_all(const vg_shape *shape, const double *x, const double *y, const double *z, const double *dx,
                 const double *dy, const double *dz, double step_max, int64_t n, int32_t *cls, double *dist_in,
                 double *dist_out, double *safety_in, double *safety_out, void *stream);

/*
 * vg_volume_create -- a mother solid holding ndaughters placed solids ("coordinate
 * transformations"; BASELINE.json configs[4]).  `xforms` (HOST): ndaughters * 12 doubles, row-major 3x4
 * [R | b] per daughter, mother -> daughter-local: p_loc = R p + b, d_loc = R d (reading R12).  R is
 * expected to be orthonormal (checked to 1e-9: VG_ERR_PARAM otherwise).  0 <= ndaughters <= VG_MAX_DAUGHTERS.
 * Mother and daughters may be any vg_shape.  With the five primitives only, ComputeStep runs the dedicated kernel (the
 * daughter table staged in shared memory by TMA); a polycone or boolean among them (reading R30) makes the volume a
 * one-level world served by the world kernels, with the same results and conventions.
 * The shapes' constants are copied; the vg_shape handles may be destroyed afterwards.
 * Built here, once, on the host and placed on the current device: the daughters' bounding spheres, the candidate grid of
 * ComputeStep and -- for 8 daughters or more -- the grid of nearest-daughter lists that vg_volume_safety reads (up to
 * 32^3 cells): about 40 ms for 64 daughters, 160 ms for 256, and 0.5 / 1.3 MiB of device memory.
 */
int vg_volume_create(const vg_shape *mother, int ndaughters, const vg_shape *const *daughters, const double *xforms,
                     vg_volume **out);
void vg_volume_destroy(vg_volume *volume); /* NULL is allowed */

/*
 * vg_compute_step -- navigation step of n tracks.
 * step: DEVICE double[n]; hit: DEVICE int32[n] in {VG_HIT_STEPMAX, VG_HIT_MOTHER, 0 .. ndaughters-1}.
 * Ties go to the lowest index, the mother first.  Tracks are expected inside the mother and outside every
 * daughter; a track outside the mother gets (-1, VG_HIT_MOTHER), a daughter the track is inside of is skipped.
 */
int vg_compute_step(const vg_volume *volume, const double *x, const double *y, const double *z, const double *dx,
                    const double *dy, const double *dz, double step_max, int64_t n, double *step, int32_t *hit,
                    void *stream);

/*
 * vg_volume_safety -- isotropic safety of the navigation state of n points (PAPER.md:113 at the level of
 * placed volumes): min( SafetyToOut_mother(p), min_i SafetyToIn_i(R_i p + b_i) ).  safety: DEVICE double[n].
 */
int vg_volume_safety(const vg_volume *volume, const double *x, const double *y, const double *z, int64_t n,
                     double *safety, void *stream);

/* ---- hierarchy of volumes ("with hierarchical connections one can build the whole detector";
 *      a particle whose geometric step wins "is transported to the border" and changes volume;
 *      SURVEY.md sec. 8(f) f3; readings R22-R25 in DESIGN.md) ----
 *
 * A world is a tree of placed solids ("nodes").  Node 0 is the root; parent[i] < i for i > 0, parent[0] = -1.
 * `xforms` (HOST): nnodes * 12 doubles, row-major 3x4 [R | b] per node, from the PARENT's local frame to the
 * node's local frame (for the root: from the world frame), orthonormal R as for vg_volume_create.  The children of
 * a node are the nodes that name it as parent, in index order; siblings must not overlap and must lie inside
 * their parent (not checked).  A node may be any vg_shape: the five primitives, a polycone or a boolean (reading R30;
 * worlds without polycone / boolean nodes run leaner kernels; with a boolean among a node and its children
 * vg_world_safety inherits the boolean's "never over-estimates" in place of "exact").  1 <= nnodes <= VG_MAX_NODES; a node has
 * at most VG_MAX_DAUGHTERS children.  The shapes' constants are copied.  The node table lives in memory of the
 * device that is current at create time.
 */
typedef struct vg_world vg_world;
#define VG_MAX_NODES 65536
int vg_world_create(int nnodes, const vg_shape *const *shapes, const int32_t *parent, const double *xforms,
                    vg_world **out);
void vg_world_destroy(vg_world *world); /* NULL is allowed */

/* vg_world_locate -- the deepest node that holds each of n points given in the world frame (R23): -1 if the point
 * is not strictly inside the root (Inside != VG_INSIDE); else descend from the root, the first child in index
 * order that holds the point strictly inside becomes the current node, until no child does.
 * node: DEVICE int32[n]. */
int vg_world_locate(const vg_world *world, const double *x, const double *y, const double *z, int64_t n,
                    int32_t *node, void *stream);

/* vg_world_step -- navigation step of n tracks, each in its own node (R24).  x..dz are in the WORLD frame;
 * node: DEVICE int32[n], the node each track is in (as vg_world_locate returns it).  The step is vg_compute_step
 * in that node (its solid as mother, its children as daughters, same tie-break); next: DEVICE int32[n] = the child
 * entered, the parent when the node's own exit wins (-1 above the root), the node itself when step_max wins.
 * A track with node outside [0, nnodes) gets (-1, -1).  step: DEVICE double[n]. */
int vg_world_step(const vg_world *world, const int32_t *node, const double *x, const double *y, const double *z,
                  const double *dx, const double *dy, const double *dz, double step_max, int64_t n, double *step,
                  int32_t *next, void *stream);

/* vg_world_safety -- vg_volume_safety in the node of each point (R25): min(SafetyToOut of the node, SafetyToIn of
 * every child); for a located point this is the distance to the nearest surface of ANY node of the world.
 * -1 for a node outside [0, nnodes).  safety: DEVICE double[n]. */
int vg_world_safety(const vg_world *world, const int32_t *node, const double *x, const double *y, const double *z,
                    int64_t n, double *safety, void *stream);

/* ---- host-buffer entry points (the scheduler hands baskets of tracks to the geometry every step;
 *      the GPU pays off once transfers are amortised) ----
 *
 * Same operations as above, but every track array and every output array is a HOST pointer (pageable or
 * pinned; pinned memory makes the copies asynchronous).  The library cuts the arrays into chunks and pipelines
 * host->device copy, the same kernels, device->host copy over several internal streams and per-device staging
 * memory allocated once on first use.  The call returns when the outputs are complete (it synchronises its own
 * streams only).  Calls on one device are serialised by a lock.  Equally spaced arrays (rows of one allocation) cross
 * the link as one strided copy per chunk; calls of up to 2^14 tracks whose arrays are all pinned run without copies
 * (the kernel addresses the pinned host memory directly).
 *
 * vg_query_host: `query` is a vg_query; out is int32[n] for VG_Q_INSIDE, double[n] otherwise; dx, dy, dz are
 * read only by the two distance queries (may be NULL otherwise), step_max likewise. */
typedef enum {
    VG_Q_INSIDE = 0,
    VG_Q_DISTANCE_TO_IN = 1,
    VG_Q_DISTANCE_TO_OUT = 2,
    VG_Q_SAFETY_TO_IN = 3,
    VG_Q_SAFETY_TO_OUT = 4
} vg_query;
int vg_query_host(const vg_shape *shape, int query, const double *x, const double *y, const double *z,
                  const double *dx, const double *dy, const double *dz, double step_max, int64_t n, void *out);
int vg_compute_step_host(const vg_volume *volume, const double *x, const double *y, const double *z, const double *dx,
                         const double *dy, const double *dz, double step_max, int64_t n, double *step, int32_t *hit);
/* vg_query_all over HOST arrays: the six track arrays cross the host link once for all five answers (48 B in,
 * up to 36 B out per track).  Outputs are HOST pointers; any may be NULL (at least one must be given). */
int vg_query_all_host(const vg_shape *shape, const double *x, const double *y, const double *z, const double *dx,
                      const double *dy, const double *dz, double step_max, int64_t n, int32_t *cls, double *dist_in,
                      double *dist_out, double *safety_in, double *safety_out);

/* vg_query_host_static -- vg_query_host for callers that must not allocate (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc; same operation as vg_query_host).  The device
 * staging area is a static array inside the library's device image (7 x VG_STATIC_MAX_TRACKS doubles = 3.5 MiB, held
 * by every GPU that loads the library until the process exits) instead of memory allocated on first use, and the call
 * makes no cudaMalloc / cudaFree / cudaHostAlloc and creates no stream or event: the host -> device copies, the same
 * kernel as the other entry points and the device -> host copy are enqueued on `stream` (a cudaStream_t, NULL = the
 * default stream) and the call returns when `out` is complete (it synchronises that stream).
 *   x, y, z (and dx, dy, dz for the two distance queries; may be NULL otherwise): HOST double[n], pageable or pinned;
 *   out: HOST int32[n] for VG_Q_INSIDE, double[n] otherwise; the caller owns every array.
 *   n > VG_STATIC_MAX_TRACKS: VG_ERR_PARAM and nothing is enqueued (split the batch, or call vg_query_host);
 *   n = 0: VG_OK, no array is touched.
 * If `stream` is being captured into a CUDA graph, the call records its copies and its kernel as nodes of that graph and
 * returns without waiting (host arrays must then be pinned, stay alive and hold the tracks at replay time; make one
 * direct call on the device before the capture, which looks up the array's address).  Replays of such graphs must not
 * overlap each other or a direct call.
 * All calls on a device share the one array: calls through this entry point are serialised by a lock and each waits
 * for its own work, so they never overlap each other, but any other way of having two of them on the GPU at once
 * (none is offered) would race.  The array keeps the previous call's contents; nothing in it needs to start at zero
 * (a call overwrites the first n elements of each array its kernel reads, and only the first n results are copied
 * out). */
#define VG_STATIC_MAX_TRACKS 65536
int vg_query_host_static(const vg_shape *shape, int query, const double *x, const double *y, const double *z,
                         const double *dx, const double *dy, const double *dz, double step_max, int64_t n, void *out,
                         void *stream);

/* ---- launch policy (process-wide; does not change any result) ----
 * VG_OPT_PIPE_MIN_N: queries over at least this many tracks whose arrays are all 16-byte aligned run as the
 * persistent TMA-pipelined kernel (track tiles staged global -> shared memory by bulk copies);
 * shorter or misaligned batches run as the plain one-pass kernel.  INT64_MAX switches the pipelined form off.
 * VG_OPT_PDL (default 1): kernels are launched with the programmatic-dependent-launch attribute, so that the launch
 * latency and set-up of a kernel overlap the tail of the previous kernel in the same stream; every kernel still
 * waits (griddepcontrol.wait) for its predecessor to complete before it touches global memory, so stream order is
 * preserved exactly.  0 launches without the attribute.
 * VG_OPT_FORM (default VG_FORM_AUTO): which of the three kernel forms a query runs as (same arithmetic, same
 * results).  DIRECT: one CTA per 512 tracks.  PIPELINED: the TMA ring above (subject to VG_OPT_PIPE_MIN_N and the
 * alignment rule).  STREAMING: one resident wave of CTAs, each owning one contiguous range of tracks and loading its
 * next pair of tracks while it evaluates the current one (16-byte aligned arrays only).  AUTO takes, per (solid,
 * query), the form that measured fastest (profiles/).
 * VG_OPT_HOST_CHUNK (default 0 = chosen from n): tracks per chunk of the host-buffer entry points' copy / compute
 * pipeline (clamped to 2^20).
 * VG_OPT_COOP_MAX_N (default VG_COOP_MAX_N_DEFAULT): queries of a full-phi polycone over at most this many tracks run as
 *   the lanes-per-track kernel (a group of 4..32 lanes shares one track and splits its sections):
 *   lowest latency for small batches, same results.  0 switches the form off, and with it the one-track-per-thread
 *   polycone kernels that serve larger batches (the persistent kernels with per-CTA staged tables run instead: the
 *   tests use this to keep every form under parity).
 * VG_OPT_NAV_FORM (default 0 = chosen per volume): how vg_compute_step evaluates the daughters that survive its cull
 *   (same results).  1: every lane walks its own candidates.  2: the candidates of a warp's 32 tracks are pooled and
 *   evaluated as one dense work list (a warp cooperates over daughters).  0 takes 2 for volumes whose candidate grid
 *   lists more than 24 daughters per cell, else 1 (DESIGN.md sec. 6.4 has the measurements). */
typedef enum { VG_OPT_PIPE_MIN_N = 0, VG_OPT_PDL = 1, VG_OPT_FORM = 2, VG_OPT_HOST_CHUNK = 3, VG_OPT_COOP_MAX_N = 4,
               VG_OPT_NAV_FORM = 5 } vg_option;
#define VG_COOP_MAX_N_DEFAULT 32768
enum { VG_FORM_AUTO = 0, VG_FORM_DIRECT = 1, VG_FORM_PIPELINED = 2, VG_FORM_STREAMING = 3 };
int vg_set_option(int option, int64_t value);
int64_t vg_get_option(int option); /* the value, or VG_ERR_ARG for an unknown option */

/* Thread-local message of the last failing call on this host thread ("" if none). Static storage. */
const char *vg_last_error(void);

/* ---- measurement helpers (used by bench.py for the roofline denominators; not part of the method) ---- */

/* Runs `launches` back-to-back launches of a register-resident chain of independent FP64 FMAs that fills the
 * device, timed with CUDA events on `stream`; writes the achieved FP64 rate in FMA instructions (lanes) per
 * second to *fma_per_s (HOST).  Synchronises the stream. */
int vg_probe_fp64_fma_rate(int launches, double *fma_per_s, void *stream);
/* Enqueues `launches` empty kernels (launch-latency floor for the small-N end of configs[3]). */
int vg_probe_empty_launch(int launches, void *stream);
/* Enqueues ONE launch of the query kernel of `query` (0 Inside, 1 DistanceToIn, 2 DistanceToOut, 3 SafetyToIn,
 * 4 SafetyToOut) instantiated with an arithmetic-free pseudo-solid: the loads, the store, the grid shape and the
 * launch form of a real query on n tracks, one add per coordinate.  Its duration is the size-matched memory ceiling
 * bench.py quotes beside the small batches.  Arrays as for the queries (dx, dy, dz unused for 0, 3, 4). */
int vg_probe_stream(int query, const double *x, const double *y, const double *z, const double *dx, const double *dy,
                    const double *dz, int64_t n, void *out, void *stream);
/* Host-only: the candidate grids vg_shape_create builds for the safeties of a polycone, recomputed
 * into caller memory so that the host logic can be checked without a device.  masks: HOST uint64[rows * cols] of the
 * surface grid; face_masks: HOST uint64[rows * 2 cols] of the phi-face grid (may be NULL); row_section: HOST
 * uint8[rows]; geom: HOST double[3] = {1 / cell width in rho, 1 / cell height in z, z of the grid's lower edge};
 * dims: HOST int[2] = {rows, cols}.  Any output pointer may be NULL.  VG_ERR_ARG if the shape is not a polycone. */
int vg_debug_polycone_grid(const vg_shape *shape, uint64_t *masks, uint64_t *face_masks, unsigned char *row_section,
                           double *geom, int *dims);
/* Host-only: the conservative cull of ComputeStep (which daughters can this ray touch?) evaluated on
 * the CPU by the very code the kernel runs (csrc/vg_nav_cull.h is compiled for both sides and rounds identically), so
 * that its soundness can be checked without a device.  mother / daughters / xforms as for vg_volume_create (primitives
 * only); x .. dz: HOST arrays of n tracks in the mother frame; t_lim: HOST array of the ray-parameter limit per track
 * (the mother's exit or the physics step; NULL = +inf); masks: HOST uint64[4 n], bit j of masks[4 i + c] set = daughter
 * 64 c + j survives for track i.  stage 0: both stages as the kernel runs them; 1: the grid walk alone; 2: the FP32
 * bounding-sphere test alone, applied to every daughter; 3: the candidates of the POINT x, y, z (the mask of its grid
 * cell, what vg_world_locate tests in a node with many children); 4: the candidates of the
 * SAFETY of the point x, y, z (the daughters that can be the nearest one anywhere in its cell of the safety grid, what
 * vg_volume_safety / vg_world_safety evaluate; every daughter outside the grid or without one).  grid: HOST double[9]
 * (stage 4: double[10]) or NULL, receives the candidate grid's origin, cell size and cells per axis (x, y, z each;
 * stage 4: the SAFETY grid's, laid over the mother's bounding box, and its cells per axis once more as the tenth
 * value; 0 = none).  No CUDA call is made. */
int vg_debug_nav_cull(const vg_shape *mother, int ndaughters, const vg_shape *const *daughters, const double *xforms,
                      const double *x, const double *y, const double *z, const double *dx, const double *dy,
                      const double *dz, const double *t_lim, int64_t n, uint64_t *masks, int stage, double *grid);
/* Host-only: a boolean as vg_boolean_create flattened it: the kinds of its primitives in tree order
 * (kinds: HOST int[8]), the 3x4 transforms from the frame of the boolean to the frame of each primitive (xforms: HOST
 * double[8 * 12]) and the postfix program (prog: HOST uint8[16]; a token < 0x80 pushes that primitive, 0x80 | op combines
 * the two on top).  Returns the number of primitives (2 for a boolean of two primitives), *nprog receives the program
 * length; VG_ERR_ARG if the shape is not a boolean.  Any output pointer may be NULL. */
int vg_debug_boolean_program(const vg_shape *shape, int *kinds, double *xforms, unsigned char *prog, int *nprog);
/* Number of kernel launches the library has made in this process (all threads). */
int64_t vg_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* VG_H */
