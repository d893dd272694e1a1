/* cel.h — C ABI of celstep, the B200-native step iteration over a struct-of-arrays array of track slots.
 *
 * What the calls are: the paper's statement of the problem (arXiv 2503.17608): a *step iteration* over a
 * large array of track slots (section 2), with the optional reindexing of slot indices
 * `state[state_indices[tid]]` (section 3.1), a cap on field substeps (section 3.3)
 * and stream-ordered memory so that the host never blocks (section 3.4), in the "standalone
 * application" model where all events are mixed in one track array. BASELINE.json's north_star
 * names the three calls cel_create / cel_transport / cel_tallies; the physics is docs/PHYSICS_SPEC.md.
 *
 * Conventions. Units: MeV, cm, tesla. All structs are plain C in HOST memory and are copied during the call
 * (the caller keeps ownership). Every call returns 0 (CEL_OK) or a negative CEL_ERR_* code; nothing throws
 * across the ABI; there is no global state; a context must be used from one host thread at a time.
 * All device work is enqueued on the context's stream (its own, or the one given by cel_set_stream).
 * There is no CPU fallback: without a CUDA device cel_create fails with CEL_ERR_CUDA.
 */
#ifndef CEL_H
#define CEL_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cel_ctx cel_ctx; /* opaque; owned by the library; freed by cel_destroy */

enum { CEL_SORT_NONE = 0, CEL_SORT_BY_ACTION = 1, CEL_SORT_BY_PARTICLE = 2,
       /* PAPER.md:51 (section 3.2): no index array; the initializers popped in an iteration are partitioned by charge and
        * assigned to opposite ends of the track array (docs/PHYSICS_SPEC.md S9-P): charged ones take the vacancies from
        * slot 0 upwards, neutral ones from slot N-1 downwards; the kernels run masked over all slots as in mode NONE */
       CEL_SORT_PARTITION = 3,
       /* PAPER.md:53 (section 3.2): reindexing by action as CEL_SORT_BY_ACTION, plus parent-slot reuse (S9-R): a slot
        * vacated by its interaction (photoelectric, pair, annihilation, a Compton photon / bremsstrahlung electron that fell
        * below the cut) takes the interaction's first secondary in place instead of pushing it to the initializer stack */
       CEL_SORT_BY_ACTION_REUSE = 4 };
enum { CEL_GEOM_SLAB = 0, CEL_GEOM_CYL = 1 };
enum { CEL_GAMMA = 0, CEL_ELECTRON = 1, CEL_POSITRON = 2 };
/* action IDs = sort keys (docs/PHYSICS_SPEC.md S2) */
enum { CEL_ACT_PE = 0, CEL_ACT_PAIR = 1, CEL_ACT_COMPTON = 2, CEL_ACT_MOVE_G = 3, CEL_ACT_MOVE_C = 4,
       CEL_ACT_BREMS = 5, CEL_ACT_ANNIH = 6, CEL_ACT_VACANT = 7 };

enum {
  CEL_OK = 0,
  CEL_ERR_INVALID_ARG = -1,   /* null pointer, bad enum, non-unit direction, primary outside the geometry, ... */
  CEL_ERR_CUDA = -2,          /* a CUDA runtime call failed (cel_last_cuda_error gives the text) */
  CEL_ERR_OOM = -3,           /* device or pinned allocation failed */
  CEL_ERR_INIT_OVERFLOW = -4, /* initializer stack exceeded init_capacity (S9); results invalid */
  CEL_ERR_TALLY_OVERFLOW = -5,/* a single deposit of 2^63 quanta (2^27 MeV) or more, or a negative one (S10); sticky, results invalid */
  CEL_ERR_NONFINITE = -6,     /* a non-finite energy, position or direction: in a device-resident primary, or produced by a step; sticky */
  CEL_ERR_NOT_RUN = -7,       /* cel_tallies before any cel_transport */
  CEL_ERR_MAX_ITER = -8,      /* the run did not end within max_iterations */
  CEL_ERR_INTERNAL = -9,      /* a bookkeeping block gave up waiting for the blocks before it (cannot happen when blocks
                                 are dispatched in index order; reported instead of hanging) */
  CEL_ERR_HIT_OVERFLOW = -10, /* more hit records in one batch of iterations than option hit_capacity (results invalid) */
  CEL_ERR_TOO_LARGE = -11     /* cel_reindex_static: more slots than its fixed device scratch holds (CEL_REINDEX_STATIC_MAX_SLOTS) */
};

/* one effective element per material (S0) */
typedef struct { double density_g_cm3, Z, A; } cel_material;

typedef struct {
  int kind;                /* CEL_GEOM_SLAB: bounds = z planes. CEL_GEOM_CYL: bounds = radii, bounds[0] = 0 (S6) */
  int n_vol;               /* 1..254 */
  const double* bounds;    /* host, n_vol+1 ascending values */
  const int* vol_material; /* host, n_vol entries, index into mats or -1 = vacuum */
  const int* vol_bin;      /* host, n_vol entries, tally bin or -1 = not scored */
  double half_x, half_y;   /* slab half-widths */
  double half_z;           /* cylinder half-length */
  double field_T[3];       /* uniform field; all zero = no field */
} cel_geometry;

typedef struct {
  uint64_t seed;           /* Philox key (S3) */
  double cut_MeV;          /* production and tracking cut; the table grid starts at 1e-3 MeV (S4) */
  int enable_pair, enable_brems, enable_msc, enable_eloss, enable_annihilation;
  int electrons_local;     /* 1 = every electron is deposited where it is born (config 1) */
  int max_substeps;        /* field substeps per iteration, 10 in the paper */
  uint32_t max_steps_per_track; /* looper kill (S7.6); 1..65535 (the step count is a 16-bit field of the slot state) */
  uint64_t init_capacity;  /* initializer stack capacity; 0 = max(8 n_slots, 2^24) */
} cel_physics;

/* 64 bytes */
typedef struct { uint32_t event; int32_t ptype; double energy_MeV; double pos[3]; double dir[3]; } cel_primary;

/* unpacked view of one track slot or one initializer (debug surface), 80 bytes */
typedef struct {
  double pos[3]; double dir[3]; double energy;
  uint32_t event; uint32_t nsteps; int32_t vol; int32_t surf; int32_t ptype; int32_t action;
} cel_track;

typedef struct {
  uint32_t n_events; int32_t n_bins;  /* bin n_bins = escaped energy */
  const uint64_t* fixed;              /* [n_events][n_bins+1], units 2^-36 MeV; library-owned pinned HOST memory,
                                         valid until the next cel_transport / cel_destroy */
  uint64_t track_steps, iterations, secondaries; /* S11 */
  double seconds;                     /* device time of the last cel_transport (CUDA events on the stream) */
  uint64_t kernel_launches;           /* kernels enqueued by the last cel_transport */
} cel_tally_view;

/* Create a context: builds the physics tables on the host (S4), uploads geometry and tables, allocates the
 * SoA state for n_slots slots (N <= 2^28), the staging areas and the initializer stack. mats: n_mats entries.
 * sort_mode: CEL_SORT_*. On success *out owns device memory until cel_destroy. */
int cel_create(const cel_geometry* geometry, const cel_material* mats, int n_mats, const cel_physics* physics,
               uint64_t n_slots, int sort_mode, cel_ctx** out);

/* Use the caller's CUDA stream (a cudaStream_t passed as void*, e.g. torch.cuda.current_stream().cuda_stream).
 * Must be called before the first cel_transport / cel_debug_begin; the stream must outlive the context. */
int cel_set_stream(cel_ctx*, void* cuda_stream);

/* Bytes of device workspace cel_create would allocate for these sizes; cel_set_workspace lets the caller own
 * that memory instead (e.g. a torch tensor): dptr is a DEVICE pointer, 256-byte aligned, bytes >= the size
 * reported; it must outlive the context and must be set before the first transport. */
uint64_t cel_workspace_bytes(uint64_t n_slots, uint64_t init_capacity, int sort_mode);
int cel_set_workspace(cel_ctx*, void* dptr, uint64_t bytes);

/* Transport: resets slots, tallies (sized n_events x (n_bins+1)) and counters, writes primary i to init[i]
 * (S9; primaries is a HOST array, validated, copied), then enqueues step iterations in batches on the stream
 * and returns when a lagged copy of the control block (written into pinned host memory by a one-warp kernel at the end of every
 * batch of iterations) shows that no track and no initializer is left.
 * The host never issues a synchronous copy or a device-wide synchronisation. */
int cel_transport(cel_ctx*, const cel_primary* primaries, uint64_t n_primaries, uint32_t n_events);

/* Same, but the primaries are already resident in DEVICE memory as n_primaries packed cel_primary records
 * (checked on the device as they are loaded: a bad event / type / volume / direction is CEL_ERR_INVALID_ARG, a non-finite or
 * non-positive energy CEL_ERR_NONFINITE, reported by the transport or the next cel_tallies); used to time the path with
 * inputs in HBM. n_events <= 2^24 in every transport call (the event id is a 24-bit field of the slot state). */
int cel_transport_device(cel_ctx*, const void* d_primaries, uint64_t n_primaries, uint32_t n_events);

/* Synchronises the stream, copies the integer tallies to pinned host memory and fills *out. */
int cel_tallies(cel_ctx*, cel_tally_view* out);

void cel_destroy(cel_ctx*);
const char* cel_strerror(int code);
const char* cel_last_cuda_error(cel_ctx*);

/* The kernels of one step iteration (S1). P1 + P2 + the iteration's counters: FILL_SORT (one pass);
 * P3i: ANNIH, PE, PAIR; P3i+P3m: PHOTON (Compton, then the photon move), CHARGED (bremsstrahlung, then the charged move
 * with energy loss and MSC); P4 (scoring) happens inside the action kernels; P5: PUSH. */
enum { CEL_K_FILL_SORT = 0, CEL_K_ANNIH, CEL_K_PE, CEL_K_PAIR, CEL_K_PHOTON, CEL_K_CHARGED, CEL_K_PUSH,
       CEL_K_PART_COUNT, CEL_K_PART_SCATTER /* the two passes of the charged / neutral partition (CEL_SORT_PARTITION) */,
       CEL_K_DISCRETE /* photoelectric + pair + annihilation in one launch (sort by action, option merge_discrete) */,
       CEL_K_HITS_FLUSH /* option hits = 1: the iteration's hit records streamed to the pinned host ring buffer */,
       CEL_K_TAIL /* small populations: one block runs whole iterations back to back (option tail) */,
       CEL_KERNEL_COUNT };
int cel_kernel_count(void);                 /* CEL_KERNEL_COUNT */
const char* cel_kernel_name(int kernel_id); /* static string, "" if out of range */
/* Per-kernel device time of the last transport run with option "profile" = 1 (per-kernel HBM
 * fractions). ms_out and launches_out are HOST arrays of CEL_KERNEL_COUNT entries: summed CUDA-event time between
 * the launch before and the launch after each kernel on the context's stream, and the number of launches timed.
 * All zero if the run was not profiled. */
int cel_kernel_times(cel_ctx*, double* ms_out, uint64_t* launches_out);

/* Run-time knobs (before a transport). use_graph: replay one captured CUDA graph per iteration (default 1).
 * batch: iterations enqueued between status polls (default 16). max_iterations: safety stop (default 2^22).
 * profile: 1 = launch the kernels directly, one after the other, with a CUDA event after each one and synchronise once
 * per batch, so that cel_kernel_times can report per-kernel device time (a measurement mode: results are identical,
 * the run is slower). concurrent: 1 (default) = the independent action kernels of an iteration run as parallel
 * branches of the iteration graph; 0 = one after the other. pdl: programmatic dependent launch along the main
 * chain (default 1). merge_discrete: photoelectric + pair + annihilation in one launch (default 1: sorted by action
 * over their three ranges, unsorted / partition as one masked pass before the move kernels; 0: one launch per action).
 * tail: 1 (default) = when the lagged status shows that live tracks + initializers fit one block (<= 512), the host enqueues
 * one single-block kernel that runs up to 256 whole iterations back to back instead of batches of the iteration graph, and
 * switches back if the population grows (the fixed cost of an iteration is exposed at low track counts);
 * results are bit-identical; not used with hits, trace, profile or CEL_SORT_PARTITION. grid_cap: blocks per SM of the action
 * kernels' grids (default 6, measured 1 % faster than 8 on config 2; several contexts sharing the GPU may take a share each).
 * live_tiles: 1 (default) = the bookkeeping kernels (fill + sort, push) walk only the leading part of the slot array that the
 * population has reached so far — vacancies are filled in ascending slot order (S9), so everything above is vacant — 0 = the
 * whole array in every iteration; results are bit-identical (always 0 on the debug surface and with CEL_SORT_PARTITION).
 * max_tiles: at most this many bookkeeping tiles (of 1024 x 2^j slots; default 0 = 1024-slot tiles up to 2^22 slots, at most
 * 8192 tiles beyond); only before the first transport, and with a caller-provided workspace the padding of the slot arrays to
 * whole tiles may need up to one tile more than cel_workspace_bytes states (INVALID_ARG then). A test and measurement knob:
 * results do not depend on it.
 * trace: see cel_trace. (Execution forms that were measured slower and removed — a persistent cooperative kernel, all
 * actions in one launch — are recorded in DESIGN.md section 10.) */
int cel_set_option(cel_ctx*, const char* name, int64_t value);

/* ---- hit transfer (section 3.4) ----
 * The paper's application hands every energy deposit ("hit") to user code on the host, so "hits must be transferred at
 * every step iteration"; doing that with synchronous copies stalled every stream, and stream-ordered
 * copies through pinned memory gave +10-100 %. cel_set_option("hits", m) before a transport:
 *   m = 1: the action kernels append one cel_hit per quantised deposit (S10; the same integers the tally receives, the
 *          escape bin included) to a device buffer; after every iteration a kernel streams the new records into one of two
 *          pinned host ring buffers (stream-ordered, no synchronisation); after each batch of iterations the host hands
 *          the previous batch's records to a consumer thread (the callback below), one batch behind the device.
 *   m = 2: the "before" of PAPER.md:67: after each batch the host waits for the stream and copies the records with a
 *          blocking cudaMemcpy on the default stream into pageable memory, then processes them inline.
 *   m = 0: off (default; the tallies are kept on the device in any mode).
 * "hit_capacity": records per batch of iterations (default 2^24 = 256 MB; more in one batch is CEL_ERR_HIT_OVERFLOW).
 * "hit_tally" = 1: the library's own consumer also accumulates the records into a host tally (cel_hit_tallies), which
 * must equal cel_tallies bit for bit (the test of the transfer). */
typedef struct { uint32_t event; int32_t bin; uint64_t q; } cel_hit;   /* 16 bytes; q in units of 2^-36 MeV; bin n_bins = escaped */
/* Called on the library's consumer thread (mode 1) or on the calling thread (mode 2), once per batch of iterations, in
 * iteration order; `hits` is library-owned memory, valid during the call. */
typedef void (*cel_hit_callback)(const cel_hit* hits, uint64_t n, void* user);
int cel_set_hit_callback(cel_ctx*, cel_hit_callback fn, void* user);
typedef struct {
  uint64_t n_hits, q_sum, bytes_d2h;  /* records received by the host in the last transport, their sum, their bytes */
  uint32_t n_events; int32_t n_bins;
  const uint64_t* fixed;              /* option hit_tally: [n_events][n_bins+1] accumulated on the host from the records
                                         (library-owned, valid until the next transport); NULL otherwise */
} cel_hit_view;
/* Synchronises the stream and waits for the consumer thread; fills *out. */
int cel_hit_tallies(cel_ctx*, cel_hit_view* out);

/* Device-side timeline (the per-iteration view of PAPER.md:81-85, fig. 2). cel_set_option("trace", n) before a
 * transport makes every kernel of the first n iterations stamp the GPU's global nanosecond timer when its first block
 * starts and when its last warp ends (two integer atomics per warp: a measurement mode, results are identical).
 * cel_trace copies the stamps to the HOST array host_out[n][CEL_KERNEL_COUNT][2] = {start_ns, end_ns} (caller-owned;
 * may be NULL to query n) and sets *n_iters = n; a kernel that did not run in an iteration (or an iteration that was
 * never reached) keeps {UINT64_MAX, 0}. cel_set_option("trace_ends", 0) stamps the starts only (no atomics at the end
 * of a kernel: the least perturbing form; end_ns stays 0). Synchronises the stream. Errors: INVALID_ARG, NOT_RUN, CUDA. */
int cel_trace(cel_ctx*, uint64_t* host_out, uint64_t* n_iters);

/* ---- reindexing without allocation (section 3.2 "state_indices"; docs/PHYSICS_SPEC.md S2) ----
 * For callers that cannot call cudaMalloc (stream capture, tight serving loops, harnesses that forbid it): the stable
 * counting sort of slot indices by action key that the transport performs in every step iteration, as ONE call that
 * allocates nothing — no cudaMalloc / cudaFree / cudaMallocAsync, no context: two kernel launches on `cuda_stream`
 * (stream-ordered; the call does not synchronise). Its per-tile histograms live in a file-scope device array of 128 KB that
 * every GPU loading the library holds until the process exits, which fixes the maximum: n_slots <=
 * CEL_REINDEX_STATIC_MAX_SLOTS (2^22), more is CEL_ERR_TOO_LARGE (nothing is launched).
 *   d_keys    DEVICE, n_slots bytes, 4-byte aligned, caller-owned: key of slot i = d_keys[i] & 7 (the action, 7 = VACANT:
 *             the low bits of the transport's key byte; higher bits are ignored)
 *   d_indices DEVICE, n_slots uint32, caller-owned, written: the slots ordered by key, ascending slot order inside a key
 *   d_offsets DEVICE, 9 uint32, caller-owned, written: offsets[k] = number of slots with a key below k (offsets[8] = n_slots)
 * All calls on one device share the scratch array: calls that may OVERLAP on the GPU (different streams, graphs in flight
 * together) race on it and must be serialised by the caller; calls on one stream are safe back to back (no state is carried
 * from call to call: every counter a call reads it has written first). The first call on a device resolves the array's
 * device address (cudaGetSymbolAddress, with the caller's current device): make it outside stream capture.
 * Errors: TOO_LARGE, INVALID_ARG (null or misaligned pointer), CUDA. */
#define CEL_REINDEX_STATIC_MAX_SLOTS (1ull << 22)
uint64_t cel_reindex_static_max_slots(void);
int cel_reindex_static(const uint8_t* d_keys, uint64_t n_slots, uint32_t* d_indices, uint32_t* d_offsets, void* cuda_stream);

/* ---- debug / parity surface (synchronous, not timed) ---- */
int cel_debug_begin(cel_ctx*, const cel_primary* primaries, uint64_t n, uint32_t n_events); /* load only */
int cel_debug_step(cel_ctx*);                                 /* exactly one step iteration, then synchronise */
int cel_debug_read_state(cel_ctx*, cel_track* host_out);      /* n_slots records */
int cel_debug_read_indices(cel_ctx*, uint32_t* idx /* n_slots */, uint32_t* offsets /* 9 */);
int cel_debug_n_initializers(cel_ctx*, uint64_t* n);
int cel_debug_read_initializers(cel_ctx*, cel_track* host_out /* n records, action = -1 */);
int cel_debug_n_counts(cel_ctx*, uint64_t* n_iterations_logged);
int cel_debug_read_counts(cel_ctx*, uint32_t* host_out /* [n][8] */);
int cel_debug_table(cel_ctx*, int material, int which /* 0 C, 1 PE, 2 pair, 3 brems, 4 range */, double* out577);
int cel_debug_uniforms(cel_ctx*, const uint32_t* slots, uint32_t n, uint32_t k, uint32_t phase, uint32_t j,
                       double* host_out);                     /* xi_j(seed, slot, k, phase) evaluated on the device */
/* The path's own elementary functions evaluated on the device, for the accuracy tests:
 * which = 0: sin x, 1: 1 - cos x for |x| <= 0.5 (the helix angle of one chord substep, S7.3: Taylor polynomials, no
 * argument reduction, no cancellation). host_in / host_out: HOST arrays of n doubles, caller-owned. */
int cel_debug_math(cel_ctx*, int which, const double* host_in, uint32_t n, double* host_out);

#ifdef __cplusplus
}
#endif
#endif /* CEL_H */
