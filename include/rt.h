/* librt.so — C ABI of the B200-native AREPO-RT subcycle (arXiv 2404.17630).
 *
 * The calls follow the paper's problem statement: the mesh is static during the subcycles, so
 * "most of the data can be transferred to the GPU once before the first subcycle and only copied
 * back after the completion of the full RT step":
 *
 *     rt_create -> rt_mesh_upload -> rt_state_init -> rt_step (many) -> rt_download -> rt_destroy
 *
 * One subcycle (Fig. 1) = thermochemistry, then two
 * Heun stages of [gradients + limiter (eqs 13-15) -> face fluxes
 * (eqs 6-10) -> apply fluxes and sources per cell].  Every step
 * runs in the library's sm_100a kernels; there is no CPU fallback.
 *
 * Conventions
 *  - fp64 everywhere; int32 cell/face ids; SoA arrays; a (k, n) array is k contiguous rows of n.
 *  - A pointer is a HOST or a DEVICE pointer as the struct's mem_kind says (all pointers of one
 *    struct alike, except where stated).  Every input pointer is borrowed for the duration of
 *    the call only; outputs are caller-allocated.  The library allocates nothing on the device
 *    except inside the caller's workspace, and never frees caller memory.
 *  - Cell order is the caller's, both ways; the library reorders cells along a Peano-Hilbert
 *    curve and faces by owner and keeps the permutation private.
 *  - Return value: 0 (RT_OK) or a negative RT_E* code; the message is in rt_last_error().
 *    No exception or abort crosses the ABI.
 *  - Calls on one context are asynchronous on the context's stream unless stated; they must be
 *    issued from one host thread at a time.
 */
#ifndef RT_H_
#define RT_H_
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RT_MAXG 8 /* maximum number of frequency groups */

enum { RT_OK = 0, RT_EINVAL = -1, RT_ENOMEM = -2, RT_ECUDA = -3, RT_ESTATE = -4, RT_EMESH = -5 };
enum { RT_MEM_HOST = 0, RT_MEM_DEVICE = 1 };
/* flags of rt_workspace_bytes: RT_WS_DEVICE_MESH = the mesh arrays handed to rt_mesh_upload are DEVICE
 * pointers (no staging space); RT_WS_ALL_FACES_CROSS = reserve flux rows for every face (needed when
 * rt_tuning asks for tiles below the default size, or when rt_mesh_upload said so in RT_ENOMEM) */
enum { RT_WS_DEVICE_MESH = 1, RT_WS_ALL_FACES_CROSS = 2 };
/* rt_mesh.right codes for boundary faces (reading S13) */
enum { RT_BC_OUTFLOW = -1, RT_BC_REFLECT = -2, RT_BC_DIRICHLET0 = -3 /* -3-k: ghost state k */ };
enum { RT_CHEM_NONE = 0, RT_CHEM_FIXED_OPACITY = 1, RT_CHEM_H_ISOTHERMAL = 2, RT_CHEM_HHE_THERMAL = 3 };

typedef struct rt_ctx rt_ctx; /* opaque, owned by the library */

/* Static unstructured mesh (per-interface left/right cell index).
 * Each face is stored once; `normal` is the unit normal pointing from `left` to `right`;
 * `fcentroid` is given in the left cell's frame (it may lie outside the box when periodic). */
typedef struct {
  int64_t ncell, nface;
  double box[3];
  int32_t periodic[3];
  int32_t mem_kind;        /* of the seven array pointers below */
  const double *volume;    /* (C)    > 0 */
  const double *centroid;  /* (3, C) geometric centroid s_i (reading S7) */
  const double *area;      /* (F)    > 0 */
  const double *normal;    /* (3, F) */
  const double *fcentroid; /* (3, F) */
  const int32_t *left;     /* (F)    in [0, C) */
  const int32_t *right;    /* (F)    in [0, C), or an RT_BC_* code */
  int32_t nghost;          /* number of Dirichlet ghost states */
  int32_t ngroup;          /* G, fixed for the life of the mesh (sizes the workspace) */
  const double *ghost_state; /* HOST (nghost, 4G): N, Fx, Fy, Fz per group */
} rt_mesh;

/* Radiation + gas state, caller's cell order. N (G, C) photon number density; F (G, 3, C) photon
 * flux; ionised fractions x_HII, x_HeII, x_HeIII (C); thermal energy density eth (C) [erg cm^-3];
 * hydrogen number density nH (C) [cm^-3] (input only; rt_download does not write it). */
typedef struct {
  int32_t mem_kind;
  int32_t pad;
  double *N, *F, *xHII, *xHeII, *xHeIII, *eth, *nH;
} rt_state;

/* Point sources S of eq (6): photons/s per group injected into `cell`. HOST. */
typedef struct {
  int32_t nsrc;
  int32_t pad;
  const int32_t *cell; /* (nsrc), caller's numbering, distinct */
  const double *rate;  /* (G, nsrc) */
} rt_sources;

typedef struct {
  int32_t ngroup;
  int32_t chem_mode;        /* RT_CHEM_* */
  int32_t order;            /* 1: piecewise constant, 2: limited linear reconstruction */
  int32_t heun;             /* 1: two-stage Heun, 0: one forward-Euler stage */
  double ctilde;            /* reduced speed of light */
  double sigma[RT_MAXG][3];    /* grey cross-sections per group for HI, HeI, HeII [cm^2] */
  double eps_heat[RT_MAXG][3]; /* photo-heating energy per absorption [erg] */
  double T_fixed;           /* H_ISOTHERMAL: temperature [K] */
  double alphaB_override;   /* > 0 replaces alpha_B(HII) */
  double y_he;              /* n_He / n_H */
  double f_accept;          /* 0.1 */
  double f_target;          /* 0.05 */
  double x_floor_rel;       /* denominator floor of relative abundance changes (S18) */
  double n_floor;           /* floor on N, ledgered as floor_added (S11) */
  int64_t max_substeps;     /* cap on chemistry attempts per cell and subcycle */
  int32_t kappa_mem_kind;
  int32_t mixed;            /* 0: fp64 throughout.  1: mixed precision ("primitive variables ... single
                             * precision, ... conserved quantities and flux summations ... double precision"): the gradient
                             * estimate, the limiter, the face states, the M1 closure and the Riemann flux in fp32 in
                             * power-of-two units; the state, the face-flux sums, the donor cap, the update, the ledgers and
                             * the chemistry in fp64.  Requires |N|, |F| < 3e38 in the caller's units.  Differs from
                             * mixed = 0 by ~1e-7 of the local state per subcycle (S28) */
  const double *kappa;      /* (C) FIXED_OPACITY only: absorption coefficient [1/length], caller's order */
} rt_params;

/* Photon budget since rt_state_init, per group, photons:
 * stored + absorbed + outflow = stored(0) + injected + inflow_bc + floor_added. */
typedef struct {
  double stored[RT_MAXG], injected[RT_MAXG], absorbed[RT_MAXG], outflow[RT_MAXG], inflow_bc[RT_MAXG],
      floor_added[RT_MAXG];
  int64_t substeps_total, substeps_max, cells_hit_cap;
  int64_t nsub_done;
} rt_ledger;

/* Optional tuning of the tile decomposition and of the launches.  Every field: 0 =
 * the library's default.  The library reads no environment variable; experiments and tests set
 * these explicitly with rt_set_tuning before rt_mesh_upload. */
typedef struct {
  int32_t tile_cells;     /* cells per gradient tile; also the upper bound of a flux tile (default 32 with
                             G >= 2, 96 with one group) */
  int32_t tile_faces;     /* owned faces per flux tile (default 240: one face per thread of a 256-thread
                             block); -1 = flux tiles of tile_cells cells each */
  int32_t tile_blocks;    /* thread blocks of the flux kernel the tile size is chosen for (default 2) */
  int32_t tile_classes;   /* 1 = off: one launch sized by the largest tile (default: two size classes) */
  int32_t flux_threads;   /* threads per block of the flux kernel (default 256) */
  int32_t grad_threads;   /* threads per block of the gradient kernel (default 4 per cell, at most 256) */
  int32_t prefetch_tiles; /* the tile kernels ask L2 for the data of the tile this many blocks ahead
                             (default 600; -1 = off) */
  int32_t chem_caps[6];   /* trial caps of the chemistry passes, 0-terminated (default 1, 8: one trial
                             for every cell, up to 8 more for the unfinished, then the rest) */
  int32_t variant;        /* bit field of experimental kernel variants (default 0) */
  int32_t reserved[9];
} rt_tuning;

/* Creates a context on CUDA device `device` issuing all work on `cuda_stream` (a cudaStream_t;
 * NULL = the legacy default stream).  The stream is borrowed and must outlive the context.
 * One context = one mesh resident on one GPU for the duration of all its subcycles (PAPER.md:232:
 * "all ... kernels run on the GPU and require the mesh ... to be available in GPU memory").
 * Errors: RT_EINVAL (out == NULL), RT_ECUDA (no such device), RT_ENOMEM (host allocation). */
int rt_create(rt_ctx **out, int device, void *cuda_stream);

/* Sets the tuning of the next rt_mesh_upload (NULL = defaults).  RT_EINVAL on out-of-range values. */
int rt_set_tuning(rt_ctx *ctx, const rt_tuning *t);

/* Bytes of device workspace rt_mesh_upload needs for this problem size (0 on invalid sizes): the
 * whole device footprint of the RT step, mesh and state (everything is held on the
 * GPU from the first subcycle to the last; the library itself allocates no device memory).
 * flags: an OR of RT_WS_* (RT_WS_DEVICE_MESH: no staging space for a host mesh, 88 bytes per face
 * less).  Without RT_WS_ALL_FACES_CROSS the workspace holds the fluxes of 0.56 nface + 1024 faces
 * that cross tile boundaries (a jittered-lattice Voronoi mesh at the default tile size has 0.54);
 * rt_mesh_upload returns RT_ENOMEM, saying so, for a mesh or a tuning that needs more. */
size_t rt_workspace_bytes(int64_t ncell, int64_t nface, int ngroup, int flags);

/* Validates the mesh (index ranges, positive volumes and areas, unit normals, closed cells:
 * |sum_f s_if A_f n_f| <= 1e-10 sum_f A_f), reorders it (Peano-Hilbert on centroids, faces by
 * owner, cell -> face lists: PAPER.md:272) and precomputes the mesh-only parts of eq (15): the
 * inverse 3x3 matrix per cell and the per-face prefactors.
 * `dev_workspace` (256-byte aligned DEVICE memory of >= rt_workspace_bytes, e.g. a torch tensor's
 * data_ptr) is borrowed until rt_destroy or the next rt_mesh_upload.  Synchronises the stream.
 * Errors: RT_EINVAL (null/sizes/alignment), RT_ENOMEM (workspace too small), RT_EMESH (validation
 * failed; message says which check), RT_ECUDA. */
int rt_mesh_upload(rt_ctx *ctx, const rt_mesh *mesh, void *dev_workspace, size_t bytes);

/* Sets parameters, sources and the initial state; resets the ledger.  `src` may be NULL.
 * This is the one host -> device transfer of the state "before the first subcycle";
 * sources are the S of eq (6).  Needs a mesh (else RT_ESTATE).  Synchronises the
 * stream (inputs are free on return).  Errors: RT_EINVAL (null pointers, ngroup != the mesh's,
 * bad chem_mode / order / controller constants, source cell out of range or listed twice),
 * RT_ECUDA. */
int rt_state_init(rt_ctx *ctx, const rt_params *p, const rt_state *s0, const rt_sources *src);

/* Individual time steps ("fluxes for interfaces with at least one active neighbour.  For
 * passive particles, only their conserved quantities are updated, taking into account the fluxes from
 * the interfaces they share with active cells"; active / passive categories that stay
 * fixed during the subcycles of one RT step).  Sets the active set of the following rt_step calls:
 * active = (C) bytes in the caller's cell order, HOST or DEVICE as mem_kind says, bit 0 = active (bit 1 marks a
 * ghost of a sharded run, see "sharded runs" below; the other bits must be zero);
 * NULL = every cell (the default, restored by rt_state_init).  A passive cell does no chemistry,
 * injects no source photons and has no gradient (reading S27); a face between two passive
 * cells carries no flux; a cell none of whose faces has an active cell is left bit for bit as it was,
 * and tiles without such cells are skipped.  Needs rt_state_init (else RT_ESTATE).  Synchronises. */
int rt_set_active(rt_ctx *ctx, int mem_kind, const uint8_t *active);

/* Advances `nsub` subcycles of length dt [same time unit as 1/ctilde * length], each in the order
 * of Fig. 1: thermochemistry with adaptive sub-steps, then two
 * Heun stages of gradients, face fluxes and their application
 * to the cells; dt obeys eq (11) and is the caller's choice.
 * Asynchronous: only enqueues kernels on the context's stream; nothing crosses the host boundary
 * inside or between subcycles.  Needs rt_state_init (else RT_ESTATE); RT_EINVAL for
 * dt <= 0 or nsub < 0; RT_ECUDA if a launch fails. */
int rt_step(rt_ctx *ctx, double dt, int nsub);

/* Copies the state (any pointer of `out` may be NULL to skip it; nH is never written) and the
 * ledger (may be NULL) out, in the caller's cell order: the transfer "after the completion of the
 * full RT step".  The ledger is the photon budget that the single-valued face fluxes
 * keep closed ("ensuring photon conservation").  Synchronises the stream.
 * Errors: RT_ESTATE (no state), RT_ECUDA. */
int rt_download(rt_ctx *ctx, rt_state *out, rt_ledger *ledger);

/* Number of kernels the context has launched since rt_create (for bench.py's gpu_launches). */
int64_t rt_kernel_launches(const rt_ctx *ctx);

/* The tile decomposition rt_mesh_upload chose, for reports: out[0] cells per tile,
 * out[1] number of tiles, out[2] largest number of face slots of a tile, out[3] faces evaluated a
 * second time because their two cells lie in different tiles, out[4] largest halo (cells outside a
 * tile that touch it) of a tile, out[5] halo cells summed over the tiles, out[6] largest per-tile
 * table in 32-bit words, out[7] all per-tile tables in 32-bit words, out[8] most owned faces of a
 * tile, out[9] largest forward halo, out[10] / out[11] dynamic shared memory (bytes) of a block of
 * the gradient / flux kernel sized for the largest tile; out[12] tiles in the flux kernel's class A
 * (run with the smaller capacities out[13] owned faces, out[14] forward halo cells and out[15] bytes
 * of shared memory; the other tiles run in a second launch).  HOST array of 16.  Needs a mesh. */
int rt_tile_info(const rt_ctx *ctx, int64_t *out);

/* Per-kernel timing with CUDA events recorded on the context's stream around every launch of
 * rt_step.  rt_profile(ctx, 1) starts recording, rt_profile(ctx, 0) stops.  rt_profile_read
 * synchronises and returns, per kernel class (0 chemistry, 1 gradient, 2 face flux, 3 update,
 * 4 ledger reduction, 5 other), the summed milliseconds and the number of launches since the last
 * read; ms and count are HOST arrays of 6.  Class 2 is k_flux (a3 and the part of a4 it finishes),
 * class 3 is k_finish (a4 for the cells with faces owned by other tiles). */
int rt_profile(rt_ctx *ctx, int enable);
int rt_profile_read(rt_ctx *ctx, double *ms, int64_t *count);

/* Where the cells went (for tests that sample by tile).  tile_of_cell: (C) int32 in the
 * caller's cell order, HOST or DEVICE as mem_kind says = the tile that owns each cell.  tile_desc: HOST
 * (T, 4) int32 with T = rt_tile_info's out[1] = per tile its owned faces, its forward halo cells, its
 * table words and the flux kernel's launch class (0 = A, 1 = B).  Either may be NULL.  Synchronises. */
int rt_debug_tiles(rt_ctx *ctx, int mem_kind, int32_t *tile_of_cell, int32_t *tile_desc);

/* Slope-limited gradients of the current state in the caller's order, DEVICE or HOST as
 * mem_kind says: gN (G, 3, C), gF (G, 3 components, 3 directions, C).  For tests. Synchronises. */
int rt_debug_gradients(rt_ctx *ctx, int mem_kind, double *gN, double *gF);

/* Advances ONE subcycle of length dt with the flux kernel of the second Heun stage recording, per
 * tile, the device clock (ns) at the start of the tile, after its tables arrived, after its data was
 * staged, after the face fluxes, after the outgoing fluxes were published, at its end, and the
 * multiprocessor and block that ran it: out = HOST array of 8 words per tile, tile-major
 * (ntile_max >= the number of tiles of rt_tile_info).  For DESIGN.md's phase timeline.  Synchronises. */
int rt_debug_tile_timeline(rt_ctx *ctx, double dt, int64_t ntile_max, uint64_t *out);

/* Micro-benchmarks of the device's fp64 pipe and shared memory (not part of the subcycle; they place
 * the ALU ceiling beside the HBM roofline).  out: HOST array of 14 = operations per
 * second of dependent-chain-free DFMA, DADD, DMUL, compare+select (max), MUFU reciprocal seed,
 * reciprocal seed + two Newton steps, MUFU rsqrt seed, IEEE division, IEEE sqrt; 16-byte
 * shared-memory loads per second with 32 distinct chunks per warp, with groups of 3 and of 8 lanes
 * reading one chunk, and with a random chunk per lane; the number of multiprocessors.  Synchronises. */
int rt_debug_alu_peak(rt_ctx *ctx, double *out);

/* The "stored" row of the photon budget, sum over cells of V_i N_(g,i) per group (the identity above rt_ledger), for
 * callers that may not allocate device memory (CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): no context, no workspace, no cudaMalloc / cudaFree / allocating library call.  The per-block partial
 * sums live in a file-scope device array of the library (4 MiB per GPU that loads it, held until the process
 * exits), sized for at most RT_NOALLOC_MAX_CELLS cells: more cells -> RT_EINVAL with a message (use rt_ledger_read
 * there).  device: CUDA device index; stream: a cudaStream_t or NULL; N_dev: DEVICE (ngroup, ncell) row-major,
 * caller's cell order; volume_dev: DEVICE (ncell); stored_dev: DEVICE (ngroup), written in stream order (the call
 * does not synchronise).  err / errlen: optional HOST buffer for the error message.  Every call on a device shares
 * the array, which keeps the previous call's contents (a call overwrites every row before reading it, nothing has
 * to be cleared): calls that overlap on the GPU - different streams without a dependency - race on it.  The first
 * call on a device looks up the array's address (cudaGetSymbolAddress): make it outside stream capture.
 * Deterministic: fixed summation order. */
#define RT_NOALLOC_MAX_CELLS (1 << 24)
int rt_stored_photons_noalloc(int device, void *stream, int64_t ncell, int ngroup, const double *N_dev,
                              const double *volume_dev, double *stored_dev, char *err, int errlen);

/* ---- sharded runs: cells in contiguous ranges of the space-filling
 * curve per GPU plus one layer of ghost cells.  PAPER.md:167: per subcycle "the primitive variables required for
 * the gradient calculations, the gradients needed for the flux calculations" are communicated; PAPER.md:258:
 * "fluxes for interfaces with cells from different MPI tasks are calculated independently on each task", so no
 * flux travels.  The library does one shard's
 * arithmetic; who talks to whom, and the transport (NCCL send/recv, peer copies), are the caller's
 * (paper_2404_17630_b200/shard.py).  A ghost is a cell of the local mesh whose rt_set_active byte has bit 1 set
 * (2 = ghost that is passive at its owner, 3 = ghost that is active there): it takes part in the fluxes of the
 * faces it shares with local cells, with the gradient its owner computed, and is never updated, does no
 * chemistry, injects nothing, and is left out of the `stored` ledger row here; the local mesh must still close
 * every ghost (the faces to cells that are not local: reflective boundary faces, which carry no ledger).
 *
 * rt_step_phase runs ONE phase of a subcycle, in order: RT_PHASE_CHEM, RT_PHASE_GRAD1, RT_PHASE_FLUX1 and, with
 * Heun, RT_PHASE_GRAD2, RT_PHASE_FLUX2 (RT_ESTATE if out of order; all five back to back are one rt_step(dt, 1),
 * bit for bit).  Between phases the caller exchanges the ghosts' rows:
 *   after CHEM and after FLUX1 (Heun): RT_HALO_U   (N, Fx, Fy, Fz) x G doubles of the buffer the next phase reads
 *   after GRAD1 and after GRAD2:       RT_HALO_GRAD 12 x G doubles (floats with rt_params.mixed) per cell
 * rt_halo_pack gathers the rows of `n` cells (cells_dev: DEVICE int32, caller's local numbering) into buf_dev
 * (DEVICE, n x rt_halo_row_bytes, 16-byte aligned); rt_halo_unpack scatters them into the ghosts.  Stream-ordered,
 * no synchronisation.  The ledger of a sharded run is the sum of the shards' ledgers. */
enum { RT_PHASE_CHEM = 0, RT_PHASE_GRAD1 = 1, RT_PHASE_FLUX1 = 2, RT_PHASE_GRAD2 = 3, RT_PHASE_FLUX2 = 4 };
enum { RT_HALO_U = 0, RT_HALO_GRAD = 1 };
int rt_step_phase(rt_ctx *ctx, double dt, int phase);
int rt_halo_pack(rt_ctx *ctx, int what, int64_t n, const int32_t *cells_dev, void *buf_dev);
int rt_halo_unpack(rt_ctx *ctx, int what, int64_t n, const int32_t *cells_dev, const void *buf_dev);
int rt_halo_row_bytes(const rt_ctx *ctx, int what);

/* Last error message of this context ("" if none); valid until the next call on it.  (No exception or
 * abort crosses the ABI: SURVEY 8(b) error convention.) */
const char *rt_last_error(const rt_ctx *ctx);

/* Frees the context (not the workspace, which is the caller's: PAPER.md:232-234 leaves the device data
 * to the caller between RT steps).  NULL is allowed. */
void rt_destroy(rt_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* RT_H_ */
