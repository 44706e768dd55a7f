/* allen_velo.h — C ABI of the B200-native VELO pixel reconstruction hot path of Allen's HLT1.
 *
 * Paper: arXiv:1912.09161, "Allen: A high level trigger on GPUs for LHCb".  Citations "P:n" are line numbers of the
 * paper text; "R<k>" are the readings of DESIGN.md §3 for points on which the paper is silent.
 *
 * Statement of the problem: "Raw detector data is copied to the GPU, the full HLT1 sequence is processed on
 * the GPU and only selection decisions and objects used for the selections, such as tracks and primary vertices, are
 * copied back"; "several thousand events at once"; no host<->device traffic besides input, output and
 * grid sizes; events are independent.  This library implements the Velo box of the sequence
 * (P:175-183): decode -> cluster -> global coordinates -> phi sort -> search by triplet -> straight-line fit ->
 * compacted outputs, for a batch of events, on one CUDA stream, without synchronising with the host.
 *
 * All functions are thread-compatible (one handle per host thread / stream).  Every pointer is marked HOST or DEVICE.
 * The caller (PyTorch in this repository) owns every device buffer, including the workspace; the handle owns only a
 * few kB of geometry constants on the device.
 */
#ifndef ALLEN_VELO_H
#define ALLEN_VELO_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- return codes (synchronous errors) ---- */
#define ALLEN_VELO_OK 0
#define ALLEN_VELO_ERR_INVALID (-1)   /* null pointer, misalignment, unsupported geometry or parameter */
#define ALLEN_VELO_ERR_CUDA (-2)      /* a CUDA runtime call failed (cudaGetLastError text via allen_velo_last_error) */
#define ALLEN_VELO_ERR_WORKSPACE (-3) /* workspace missing, or too small for the per-event tables of n_events plus a minimal slab */

/* ---- per-event status bits (asynchronous conditions, written to clusters.status[e]; R8) ---- */
#define ALLEN_VELO_STATUS_BAD_HEADER 1u         /* magic / bank count / sizes / offsets inconsistent: event skipped */
#define ALLEN_VELO_STATUS_BAD_SP 2u             /* an SP word addressed a pixel outside the sensor: word ignored */
#define ALLEN_VELO_STATUS_TOO_MANY_CLUSTERS 4u  /* > 65535 clusters: clusters written, tracking skipped */
#define ALLEN_VELO_STATUS_CLUSTER_CAPACITY 8u   /* out_clusters.capacity exceeded: this event's clusters (and tracks) are not written */
#define ALLEN_VELO_STATUS_TRACK_CAPACITY 16u    /* out_tracks capacities exceeded: this event's tracks not written */
#define ALLEN_VELO_STATUS_STAGE_OVERFLOW 32u    /* a staging capacity was exceeded: event incomplete.  > 8192 SP words in one
                                                 * layer: that layer's clusters are missing; > 1024 clusters in one layer (or a
                                                 * workspace smaller than allen_velo_workspace_bytes()): clusters written, no tracks */

/* Cuts of the track search (R5).  The defaults are allen_velo_default_params(). */
typedef struct {
  int32_t w_seed_phi16; /* half-width of the seeding phi window, in phi16 units (2*pi/65536 rad); default 512 */
  int32_t w_fwd_phi16;  /* half-width of the forwarding phi window; default 512; both must be in [0, 16383] */
  float max_slope;      /* |tx|,|ty| limit of the seed's first segment; default 0.4 */
  float s_seed;         /* scatter cut for seeds, mm^2; default 2^-6 */
  float s_fwd;          /* scatter cut for forwarding, mm^2; default 2^-4 */
  float s_weak;         /* three-hit tracks are kept only if their seed scatter <= s_weak; default 2^-7 */
  int32_t max_skipped;  /* consecutive layers a track may miss before it is closed; default 1 */
} allen_velo_params_t;

/* Detector description (R1, R4; "26 planes of silicon pixel sensors").  HOST pointers, copied at create. */
typedef struct {
  uint32_t n_sensors;            /* = number of raw banks per event; <= 4096 */
  uint32_t n_modules;
  uint32_t n_layers;             /* 3 <= n_layers <= 64; at most 8 sensors per layer */
  uint32_t n_cols, n_rows;       /* pixels per sensor; n_cols even <= 1024, n_rows multiple of 4 <= 256,
                                    n_cols*n_rows <= 2^18 */
  float pitch_mm;
  const uint16_t* sensor_module; /* HOST [n_sensors] */
  const uint16_t* module_layer;  /* HOST [n_modules]; layers are numbered by increasing z */
  const float* sensor_ltg;       /* HOST [n_sensors][9] row-major local->global: (x,y,z) = M * (u, v, 1) */
  allen_velo_params_t params;
} allen_velo_geometry_t;

/* Cluster output (A2-A4, A9 of SURVEY §8(a)): compacted structure of arrays on the DEVICE.
 * Normative order inside an event: ascending (layer, phi16 as signed, key).  `capacity` = number of clusters the
 * per-cluster arrays can hold.  event_offsets/layer_offsets always report the true totals. */
typedef struct {
  uint32_t capacity;
  uint32_t* event_offsets; /* DEVICE [n_events+1]            first cluster of every event */
  uint32_t* layer_offsets; /* DEVICE [n_events*n_layers+1]   first cluster of every (event, layer) */
  uint32_t* key;           /* DEVICE [capacity] (sensor << 18) | min over pixels of (row*n_cols + col) */
  uint32_t* n_pixels;      /* DEVICE [capacity] */
  uint32_t* sum_col;       /* DEVICE [capacity] integer centroid sums (R2) */
  uint32_t* sum_row;       /* DEVICE [capacity] */
  float* x;                /* DEVICE [capacity] global position, mm (R3) */
  float* y;
  float* z;
  int16_t* phi16;          /* DEVICE [capacity] round(atan2(y,x) * 32768/pi) by the normative polynomial (R3) */
  uint32_t* checksum;      /* DEVICE [capacity] or NULL: sum of mix32(pixel) over the cluster's pixels (R2) */
  uint32_t* status;        /* DEVICE [n_events] ALLEN_VELO_STATUS_* bits */
} allen_velo_clusters_t;

/* Track output (A5-A9).  hits[] are event-local cluster indices in the normative cluster order, listed in order of
 * addition (seed a, b, c, then forwarded hits: strictly decreasing layers).  Tracks of an event appear in order of
 * creation (iteration i = L-1..2, then ascending middle hit). */
typedef struct {
  uint32_t capacity_tracks;
  uint32_t capacity_hits;
  uint32_t* event_offsets; /* DEVICE [n_events+1]        first track of every event */
  uint32_t* hit_offsets;   /* DEVICE [capacity_tracks+1] first entry of hits[] of every track; the last element
                              [capacity_tracks] always receives the total number of hits of the batch (the value
                              hit_offsets[n_tracks] has when the tracks fit), also when TRACK_CAPACITY is flagged; the
                              entries of the tracks that are written, and the end of the last of them, are valid */
  uint16_t* hits;          /* DEVICE [capacity_hits] */
  float* x0;               /* DEVICE [capacity_tracks] straight-line fit x(z) = x0 + tx*z, y(z) = y0 + ty*z (R6) */
  float* y0;
  float* tx;
  float* ty;
  float* kalman;           /* DEVICE [capacity_tracks][12] or NULL: simple Kalman fit (R9) at the track's last hit
                              (the most upstream one): x, y, tx, ty, z, chi2, then the covariances C00, C01, C11 of
                              (position, slope) for x and for y */
} allen_velo_tracks_t;

/* Primary vertices (R10; optional, beyond the headline path): a fixed number of slots per event. */
typedef struct {
  uint32_t max_per_event; /* slots per event in `vertices`; at most 32 are ever filled */
  uint32_t* n_vertices;   /* DEVICE [n_events] */
  float* vertices;        /* DEVICE [n_events][max_per_event][8]: x, y, z, sum of track weights, tracks with weight > 0,
                             chi2 (sum w chi2_t), z of the histogram seed, 0 */
} allen_velo_vertices_t;

typedef struct allen_velo allen_velo_t;

/* Fills *params with the default cuts of R5. */
void allen_velo_default_params(allen_velo_params_t* params /* HOST out */);

/* Creates a handle for the current CUDA device and copies the geometry to it.  Returns ALLEN_VELO_OK or
 * ALLEN_VELO_ERR_INVALID (unsupported geometry / parameters) / ALLEN_VELO_ERR_CUDA. */
int allen_velo_create(const allen_velo_geometry_t* geometry /* HOST */, allen_velo_t** out /* HOST out */);

/* Upper bound of the scratch memory reconstruct() needs for a batch of n_events whose raw data take raw_bytes
 * (0 if n_events * n_layers >= 2^31: such a batch is refused).  reconstruct() itself cannot know raw_bytes (the offsets
 * are on the device): it returns ALLEN_VELO_ERR_WORKSPACE only if the workspace cannot hold the tables that scale with
 * n_events plus a minimal slab; with a workspace smaller than this bound the events whose clusters do not fit the slab
 * are flagged STAGE_OVERFLOW, nothing is written out of bounds. */
size_t allen_velo_workspace_bytes(const allen_velo_t* handle, uint32_t n_events, size_t raw_bytes);

/* Registers a caller-owned DEVICE buffer (256-byte aligned) as workspace for subsequent reconstruct() calls. */
int allen_velo_set_workspace(allen_velo_t* handle, void* dev_ptr /* DEVICE */, size_t bytes);

/* Optional: average number of SP words per (event, layer) of the batches to come (raw bytes / 4 / n_events / n_layers is
 * close enough).  The results never depend on it; it selects the cluster-kernel instance whose shared-memory
 * capacity suits the occupancy (above 192 words per layer: 512 entries per layer instead of 256).  0 = no hint. */
int allen_velo_set_occupancy_hint(allen_velo_t* handle, uint32_t sp_words_per_layer);

/* Optional: the local clustering variant of P:179 ("a clustering algorithm employing bit masks, which searches for
 * clusters locally in small regions. Every region can be treated independently"; R11).  From now on a cluster
 * is a maximal 8-connected set of fired pixels INSIDE one region of sp_cols x sp_rows super-pixels (powers of two; the
 * regions tile every sensor from its pixel (0, 0)): clusters that cross a region border are split there.  (0, 0)
 * switches back to exact connected components, the default and the definition the headline path is graded on.
 * Everything downstream (positions, sort, tracks) is computed from the clusters of the chosen variant. */
int allen_velo_set_cluster_regions(allen_velo_t* handle, uint32_t sp_cols, uint32_t sp_rows);

/* Optional: from now on reconstruct() also finds primary vertices and writes them to `out` (a HOST struct of DEVICE
 * pointers, copied; NULL switches it off again).  Needs out_tracks->kalman in the reconstruct() calls (the vertex fit
 * uses the Kalman states); reconstruct() returns ALLEN_VELO_ERR_INVALID otherwise. */
int allen_velo_set_vertex_output(allen_velo_t* handle, const allen_velo_vertices_t* out);

/* Enqueues the whole hot path for one batch on `cuda_stream` and returns WITHOUT synchronising.
 *   raw_banks      DEVICE, 16-byte aligned: events in raw format v1 (R1) back to back
 *   event_offsets  DEVICE [n_events+1]: byte offset of every event in raw_banks, multiples of 16
 *   cuda_stream    a cudaStream_t (NULL = legacy default stream)
 *   out_clusters / out_tracks  HOST structs of DEVICE pointers; outputs are valid once the stream reaches this point.
 * The call only enqueues kernels, memsets and event waits (the larger search instances run on streams owned by the
 * handle that fork from and join `cuda_stream`); it allocates nothing and never waits for the device, so it may be
 * captured in a CUDA graph (stream capture on `cuda_stream`) and replayed on new contents of the same buffers.
 * Returns ALLEN_VELO_OK, ALLEN_VELO_ERR_INVALID, ALLEN_VELO_ERR_WORKSPACE or ALLEN_VELO_ERR_CUDA (launch failure). */
int allen_velo_reconstruct(allen_velo_t* handle, const void* raw_banks, const uint32_t* event_offsets,
                           uint32_t n_events, void* cuda_stream,
                           const allen_velo_clusters_t* out_clusters, const allen_velo_tracks_t* out_tracks);

/* Text of the last CUDA error seen by this handle ("" if none).  HOST string owned by the handle. */
const char* allen_velo_last_error(const allen_velo_t* handle);

void allen_velo_destroy(allen_velo_t* handle);

#ifdef __cplusplus
}
#endif
#endif /* ALLEN_VELO_H */
