/* cbm_trigger.h -- C ABI of libcbmtrigger.so
 *
 * B200-native (sm_100a) first-level J/psi -> mu+ mu- event selection for the CBM muon
 * chambers (MUCH), after Singhal, Chattopadhyay, Friese, "Investigation of heterogeneous
 * computing platforms for real-time data analysis in the CBM experiment" (arxiv 1810.11966;
 * PAPER.md).  Plain C: plain pointers and sizes, no exceptions and no C++/torch types cross
 * this boundary.  Every pointer argument says HOST or DEVICE.
 *
 * What is computed (section 3.2 steps 1-3, with the integer slope windows and
 * the cross-station linking BASELINE.json's north_star fixes):
 *
 *   compat(h in layer A, g in layer B; a/b) :=  b*|x_h*z_B - x_g*z_A| <= a*z_A*z_B
 *                                           and b*|y_h*z_B - y_g*z_A| <= a*z_A*z_B       (int64, exact)
 *   T_s  := { (h0,h1,h2) in layer0 x layer1 x layer2 of station s : all three pairs compat under win_in }
 *           -- PAPER.md:73 "Create all possible triplets of hits ..., with one hit from each layer";
 *              the triplet and the event vertex (0,0) lie on a straight line in x-z and y-z
 *   link(t in T_s, u in T_{s+1}) := compat(t.h1, u.h1; win_link)            (middle-layer hits)
 *   candidates := number of tuples (t_0, ..., t_{S-1}), t_s in T_s, consecutive ones linked
 *   n_triplets[e*S+s] = min(2^32-1, |T_s|);  n_candidates[e] = min(2^32-1, candidates)
 *   accept[e] = n_candidates[e] >= min_candidates        -- PAPER.md:88 "Select the event if it contains at
 *                                                            least two triplets ..." (generalised to candidates)
 *
 * Data layout ("separate data containers for each coordinate axis", one record per batch):
 *   x[n_hits], y[n_hits]   int32, 10-um units; hits of event e, layer l (= 3*station + layer-in-station)
 *                          are x[off[e*L+l] .. off[e*L+l+1]);  z is a per-layer constant (config)
 *   off[n_events*L + 1]    uint32, off[0] = 0, non-decreasing, off[n_events*L] = n_hits, L = 3*n_stations
 *
 * Error behaviour: every call returns CBM_OK (0) or a negative code; on error nothing is enqueued and the
 * handle stays usable.  cbm_trigger_last_error() returns a handle-owned message for the last failure.
 * A handle is not thread-safe; different slots may be driven from one thread as a software pipeline.
 *
 * Arithmetic range: the device evaluates |x_h*z_B - x_g*z_A| <= floor(a*z_A*z_B/b) in int64, which is exact
 * for any int32 x, y and 0 < z <= 2^23 (|D| < 2^56); no coordinate-range check is needed or made.
 *
 * Where input errors are found (reading B1): upload_events checks O(1) facts on the host (capacity,
 * off[0] == 0, off[n_events*L] == n_hits); the O(E*L) structural checks (offsets non-decreasing and <= n_hits,
 * no layer above max_hits_per_layer) run on the device inside `run` (classify_kernel reads off[] anyway) and are
 * reported by fetch_results / device_status as CBM_ERR_RANGE.
 */
#ifndef CBM_TRIGGER_H
#define CBM_TRIGGER_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CBM_TRIGGER_MAX_STATIONS 8
#define CBM_TRIGGER_MAX_LAYERS 24
#define CBM_TRIGGER_MAX_HITS_PER_LAYER 4096
#define CBM_TRIGGER_MAX_SLOTS 4
#define CBM_TRIGGER_N_KERNELS 6 /* classify, tile, class M, class H, class G, list X (see cbm_trigger_stats_t) */
#define CBM_TRIGGER_MAX_INDEX 0xFFFFE000u /* 2^32 - 8192: largest element count of the device-side scans (records of
                                             a stream, max_events * layers + 1); their uint32 block arithmetic (blocks of
                                             4096 elements) cannot wrap below it */
#define CBM_TRIGGER_PROFILE_RING 32 /* run_device calls whose per-kernel times are kept (CBM_FLAG_PROFILE) */

enum {
  CBM_OK = 0,
  CBM_ERR_INVALID_ARG = -1, /* null pointer, bad struct_size, S out of range, z not positive/increasing, den = 0 */
  CBM_ERR_RANGE = -2,       /* offsets not monotone / beyond n_hits, a layer above max_hits_per_layer (found on
                               the device during run, reported by fetch_results / device_status) */
  CBM_ERR_CAPACITY = -3,    /* n_events / n_hits beyond the capacity given at create */
  CBM_ERR_STATE = -4,       /* run before upload, fetch before run, slot out of range */
  CBM_ERR_CUDA = -5         /* CUDA runtime failure (no device, out of memory, launch failure) */
};

typedef struct cbm_trigger cbm_trigger_t; /* opaque; owned by the caller via create/destroy */

typedef struct {
  uint32_t struct_size;  /* = sizeof(cbm_trigger_config_t) */
  uint32_t n_stations;   /* S, 1..8; three layers per station */
  int32_t  layer_z[CBM_TRIGGER_MAX_LAYERS]; /* z of layer 3*s+l, 10-um units, 0 < z <= 2^23, strictly increasing */
  uint32_t win_in_num, win_in_den;     /* in-station slope window a/b (half-width, closed); 0 < den <= 4096, num <= den */
  uint32_t win_link_num, win_link_den; /* cross-station window a/b, same limits */
  uint32_t min_candidates;             /* accept iff n_candidates >= this (2) */
  uint32_t max_events;                 /* capacity of one slot, in events; max_events * 3 * n_stations + 1 <= CBM_TRIGGER_MAX_INDEX */
  uint64_t max_hits;                   /* capacity of one slot, in hits; < 2^32 */
  uint32_t max_hits_per_layer;         /* 1..4096; an event with a fuller layer is rejected (CBM_ERR_RANGE) */
  uint32_t n_slots;                    /* 0..4 slots of (pinned host + device) buffers; 2 = double buffering.
                                          0: only cbm_trigger_run_device() is usable (caller owns all buffers) */
  int32_t  device;                     /* CUDA ordinal */
  uint32_t tiny_max_layer_hits;        /* tuning: events whose fullest layer holds <= this many hits (and that fit
                                          the tile) take the thread-per-station path. 0 = default (24); max 32 */
  uint32_t flags;                      /* CBM_FLAG_* */
} cbm_trigger_config_t;

#define CBM_FLAG_PROFILE 1u      /* record CUDA events around every kernel (cbm_trigger_get_stats: kernel_ms) */
#define CBM_FLAG_NO_TINY_PATH 2u /* tuning/testing: route every event through the team kernels */
#define CBM_FLAG_PACKED_INPUT 4u /* the slots take the packed wire format XY20 (cbm_trigger_upload_events_packed) */
#define CBM_FLAG_SERIAL 8u       /* measuring: launch the kernels of a run one after the other on one stream instead of
                                    side by side, so that kernel_ms are kernel times (results are identical) */

typedef struct {
  uint32_t struct_size;
  uint32_t n_events;
  uint64_t n_hits;
  uint32_t n_class[4];     /* events handled by: [0] tile kernel (tiny), [1] team_M, [2] team_H, [3] team_G */
  uint32_t n_redone;       /* events one of those kernels handed on (a shared-memory table overflowed); redone by team_X */
  uint32_t n_invalid;      /* events rejected on the device (bad offsets / layer too full); their outputs are 0 */
  uint32_t first_invalid;  /* smallest such event index, 0xFFFFFFFF if none */
  uint32_t n_launches;     /* kernels launched by the last run of this slot */
  float    kernel_ms[CBM_TRIGGER_N_KERNELS]; /* CBM_FLAG_PROFILE only: device time of classify_kernel, tile_kernel,
                                                 team_kernel (class M), chain_kernel (class H), team_kernel (class G),
                                                 team_kernel (list X) (CUDA events on the stream of each), else 0.  Without
                                                 CBM_FLAG_SERIAL the kernels share the GPU, so a time includes waiting */
  float    h2d_ms, d2h_ms; /* CBM_FLAG_PROFILE only */
} cbm_trigger_stats_t;

/* Creates a handle: validates cfg (CBM_ERR_INVALID_ARG before any CUDA call), selects cfg->device, allocates
 * n_slots x (pinned HOST staging + DEVICE arrays + result buffers) and the scheduler's device scratch, creates
 * the H2D / compute / D2H streams.  *out is written only on success.  cfg: HOST. */
int cbm_trigger_create(const cbm_trigger_config_t* cfg, cbm_trigger_t** out);

/* Frees everything the handle owns (waits for its streams first).  NULL is allowed. */
void cbm_trigger_destroy(cbm_trigger_t* h);

/* Zero-copy staging: HOST pointers into the slot's pinned buffers (owned by the handle; capacity max_hits int32
 * for x and y, max_events*L+1 uint32 for off).  A producer (DAQ / generator) writes a batch there and then calls
 * upload_events with these same pointers, which skips the staging memcpy.  (data are delivered
 * into host memory, then transferred.)
 * Contract: between upload_events(slot) and the next fetch_results(slot) the slot's host buffers are the source of
 * an H2D copy that may still be in flight: the producer must not write them in that interval (upload_events
 * itself waits for the slot's previous copy before it touches them).  The handle's compute-side streams and
 * fork/join events are shared by all slots and by run_device: runs of one handle are serialised on the device. */
int cbm_trigger_host_buffers(cbm_trigger_t* h, uint32_t slot, int32_t** x, int32_t** y, uint32_t** off);

/* a1+a2: enqueue the H2D copy of one batch into `slot` on the slot's copy stream.
 * x, y: HOST, n_hits int32 each.  off: HOST, n_events*L+1 uint32 (layout above).  If the pointers are not the
 * slot's own pinned buffers, the data are first memcpy'd into them, so caller memory may be reused on return.
 * Checks on the host, O(1): capacity, off[0] == 0, off[n_events*L] == n_hits.  The O(E*L) structural checks
 * (monotone offsets, per-layer cap) run on the device inside `run`.  Waits for the slot's previous use.
 * PAPER.md:160-161 "allocate memory on the device ... transfer the data from host to device". */
int cbm_trigger_upload_events(cbm_trigger_t* h, uint32_t slot, uint32_t n_events, uint64_t n_hits,
                              const int32_t* x, const int32_t* y, const uint32_t* off);

/* Packed wire format XY20 (shrinking the transfer was the paper's biggest
 * win): 5 bytes per hit instead of 8.  xy20[5*i .. 5*i+4] holds hit i of x[] / y[], little endian: bits 0..19 = x,
 * bits 20..39 = y, each 20-bit two's complement (10-um units, -524288 <= v <= 524287; a producer with larger
 * coordinates must use the int32 format).  A handle created with CBM_FLAG_PACKED_INPUT stages and copies the
 * packed stream (n_hits*5 bytes, rounded up to 20) and `run` first expands it on the device into the int32
 * arrays the kernels read; results are identical to uploading the same hits as int32.  Such a handle accepts
 * only the packed calls (the int32 ones return CBM_ERR_STATE) and vice versa.  Otherwise as
 * cbm_trigger_host_buffers / cbm_trigger_upload_events.  xy20: HOST (capacity max_hits*5 bytes), off: HOST. */
int cbm_trigger_host_buffers_packed(cbm_trigger_t* h, uint32_t slot, uint8_t** xy20, uint32_t** off);
int cbm_trigger_upload_events_packed(cbm_trigger_t* h, uint32_t slot, uint32_t n_events, uint64_t n_hits,
                                     const uint8_t* xy20, const uint32_t* off);

/* The producer side of XY20, for a C caller (host code, no CUDA, no handle): writes hit i of x[] / y[] (HOST, int32)
 * to out[5*i .. 5*i+4] (HOST, n_hits*5 bytes; may be a slot's buffer from cbm_trigger_host_buffers_packed).
 * Returns CBM_OK, CBM_ERR_INVALID_ARG for a NULL pointer with n_hits > 0, or CBM_ERR_RANGE if a coordinate lies
 * outside [-524288, 524287]: then *first_bad (HOST, may be NULL) is the smallest such hit index and the bytes of the
 * hits before it have been written.  On success *first_bad is n_hits. */
int cbm_trigger_pack_xy20(const int32_t* x, const int32_t* y, uint64_t n_hits, uint8_t* out, uint64_t* first_bad);

/* a3-a8: enqueue the selection kernels for the batch in `slot` after its H2D, and the D2H of the results after
 * the kernels (separate streams, event-ordered).  Returns immediately.
 * PAPER.md:162-163 "launch the kernel ... events are processed in parallel". */
int cbm_trigger_run(cbm_trigger_t* h, uint32_t slot);

/* a9: blocks until the slot's results are in pinned host memory, then copies them to the caller's HOST arrays:
 * n_triplets[n_events*S] (may be NULL), n_candidates[n_events], accept[n_events] (may be NULL).
 * Returns CBM_ERR_RANGE if the device rejected any event (outputs of those events are 0, all others are valid;
 * last_error names the first one).  PAPER.md:164 "the list of selected events is transferred back". */
int cbm_trigger_fetch_results(cbm_trigger_t* h, uint32_t slot, uint32_t* n_triplets, uint32_t* n_candidates,
                              uint8_t* accept);

/* The list of selected events ("the list of selected events is transferred back to the host"):
 * the ids of the events of the slot's last run with accept != 0, in ascending order (so the list is unique),
 * built on the device by an order-preserving compaction of accept[] as part of `run`.  Blocks until the run's
 * results are on the host.  event_ids: HOST, room for `capacity` uint32; n_selected: HOST, always written.
 * Returns CBM_ERR_CAPACITY (and writes only *n_selected) if more than `capacity` events were selected,
 * CBM_ERR_STATE without a preceding run.  May be called before or after fetch_results, until the next upload. */
int cbm_trigger_fetch_selected(cbm_trigger_t* h, uint32_t slot, uint32_t* event_ids, uint32_t capacity,
                               uint32_t* n_selected);

/* The same compaction on caller-owned DEVICE arrays on the caller's stream (see cbm_trigger_run_device):
 * d_accept[n_events] uint8 in; d_event_ids (room for n_events uint32) and d_n_selected (one uint32) out.
 * Asynchronous; uses the handle's scheduler scratch, so calls on one handle must be stream-ordered. */
int cbm_trigger_select_device(cbm_trigger_t* h, uint32_t n_events, const uint8_t* d_accept, uint32_t* d_event_ids,
                              uint32_t* d_n_selected, void* stream);

/* The list of selected events for callers that must not allocate device memory.
 *
 * Who needs it: a readout node that runs the selection inside its data-taking loop.  Such a node hands out all of its
 * device memory once, at start of run (timeslice buffers, result rings), and from then on nothing in the loop may call
 * cudaMalloc / cudaFree: both stall every stream of the device until they return, which breaks the overlap of
 * transfer and computation the loop lives on, and on a card that is fully handed out they simply fail.
 * The same holds for code that is plugged into somebody else's framework and only receives device pointers and a
 * stream from it.  Every other entry point of this library needs a handle, and cbm_trigger_create allocates.  This one
 * takes no handle and allocates nothing, neither on the device nor on the host, neither here nor in a library routine.
 *
 * What it does: exactly cbm_trigger_select_device -- d_accept[n_events] uint8 in; out: d_event_ids
 * (room for n_events uint32) = the ids of the events with accept != 0, ascending, and *d_n_selected (one uint32) =
 * their number; all three DEVICE, owned by the caller; elements of d_event_ids beyond the count are left alone.  It
 * runs on the calling thread's CURRENT device, on `stream` (a cudaStream_t of that device passed as void*; NULL = the
 * legacy default stream), and returns without waiting.
 *
 * The price: the per-block counts of the compaction live in one fixed array inside the library's device image
 * (CBM_TRIGGER_NOALLOC_MAX_EVENTS / 4096 uint32 = 16 KB).  Every GPU that loads the library carries these 16 KB until
 * the process ends, whether the call is used or not.  n_events above CBM_TRIGGER_NOALLOC_MAX_EVENTS is refused with
 * CBM_ERR_CAPACITY before anything is enqueued (split the batch, or use a handle).
 * There is one such array per device and every call on that device uses it.  Nothing in it has to be zero at the
 * start: each call first writes every entry it later reads, so the previous call's contents do no harm.  But two calls
 * that run on the GPU at the same time (different streams without an event between them, or two host threads) overwrite
 * each other's counts and both results are garbage: order the calls on one device yourself.  Calls on different
 * devices are independent.
 *
 * First call on a device: it looks up where the driver put the array on that device and keeps the address (host
 * side, a few bytes, under a lock); with lazy module loading this is also when the driver brings the two kernels onto
 * the device.  Make that first call during set-up, outside any stream capture; later calls only launch kernels.
 *
 * Errors (message from cbm_trigger_last_error(NULL), per thread): CBM_ERR_INVALID_ARG for a NULL pointer,
 * CBM_ERR_CAPACITY as above, CBM_ERR_CUDA if the device lookup or a launch fails.  Nothing is enqueued on error. */
#define CBM_TRIGGER_NOALLOC_MAX_EVENTS (1u << 24)
int cbm_trigger_select_noalloc(uint32_t n_events, const uint8_t* d_accept, uint32_t* d_event_ids, uint32_t* d_n_selected,
                               void* stream);

/* The hits of the selected events as a compact batch (the selected events go
 * on to full track reconstruction), on caller-owned DEVICE arrays on the caller's stream.  In: the batch
 * (d_x, d_y, d_off as in cbm_trigger_run_device) and the list from cbm_trigger_select_device (d_event_ids,
 * *d_n_selected: the count is read on the device, no host synchronisation).  Out, same layout restricted to the
 * selected events in list order: d_out_off[n_selected*L + 1] (starts at 0; room for n_events*L + 1 uint32),
 * d_out_x / d_out_y (room for all n_hits int32 in the worst case), *d_out_n_hits (uint64) = hits gathered.
 * No atomics: the output is unique.  Asynchronous; uses the handle's scratch (stream-ordered calls only).
 * The list is not trusted: at most n_events entries are read, and an id >= n_events or an event whose offsets
 * off[e*L .. e*L+L] are not non-decreasing inside [0, n_hits] is gathered as an empty event.  A list that names
 * an event more than once can gather more than n_hits hits: then *d_out_n_hits (> n_hits) reports the total (summed
 * in 64 bits: 2^32 hits and more are reported as they are) and nothing else is written. */
int cbm_trigger_gather_device(cbm_trigger_t* h, uint32_t n_events, uint64_t n_hits, const int32_t* d_x, const int32_t* d_y,
                              const uint32_t* d_off, const uint32_t* d_event_ids, const uint32_t* d_n_selected,
                              int32_t* d_out_x, int32_t* d_out_y, uint32_t* d_out_off, unsigned long long* d_out_n_hits,
                              void* stream);

/* The input filter of the paper's implementation "i3" ("we introduced a
 * filtering of the data ..., such that only hit data in the trigger station are transferred"), for a full-setup
 * hit stream that lies on the DEVICE: d_xyz holds n_records records (x, y, z) of int32 (10-um units; the layout of
 * PAPER.md:166-170), d_ev_off[n_events + 1] (uint32, non-decreasing, last = n_records) the records of every event.
 * A record is a hit of layer l iff its z equals the handle's layer_z[l]; all other records (other detectors) are
 * dropped.  Output: the batch layout above -- d_out_off[n_events*L + 1], and in d_out_x / d_out_y (room for n_records
 * int32 in the worst case, 16-byte aligned and padded as for cbm_trigger_run_device) the kept hits of every event
 * grouped by layer, in stream order inside a layer (so the output is unique) -- ready for cbm_trigger_run_device on
 * the same stream.  An event with ev_off[e] > ev_off[e+1] or beyond n_records keeps nothing.  Asynchronous; no
 * atomics on global memory; uses the handle's scratch (stream-ordered calls only).  n_records <= CBM_TRIGGER_MAX_INDEX, else
 * CBM_ERR_CAPACITY. */
int cbm_trigger_filter_device(cbm_trigger_t* h, uint32_t n_events, uint64_t n_records, const int32_t* d_xyz,
                              const uint32_t* d_ev_off, int32_t* d_out_x, int32_t* d_out_y, uint32_t* d_out_off, void* stream);

/* Event building from a free-streaming, time-stamped hit stream (section 8: the
 * data acquisition "will deliver free-streaming data not associated to single event by a hardware trigger ... not only
 * the spatial coordinates, but also the time measurement of each hit must be considered").  The paper states no rule;
 * DESIGN.md reading B9 fixes one: the records of a timeslice come in stream order, d_t[i] (DEVICE, int32, any unit,
 * e.g. ns from the start of the timeslice) is the time stamp of record i -- the fourth coordinate of the records
 * (x, y, z) of cbm_trigger_filter_device, kept as a container of its own.  Record i opens a new event
 * iff i == 0 or d_t[i] - d_t[i-1] > t_gap (exact 64-bit difference; a record earlier than its predecessor never opens
 * one: stream order rules); an event is a maximal run of records without such a gap, so interactions closer than t_gap
 * pile up into one event.  Output: d_ev_off (DEVICE, room for n_records + 1 uint32): d_ev_off[k] = first record of
 * event k, d_ev_off[*n_events] = n_records -- the d_ev_off argument of cbm_trigger_filter_device, whose output goes to
 * cbm_trigger_run_device.  *n_events (HOST) = number of events built.  Blocks until the count is on the host (the next
 * calls need it as an argument); n_records <= CBM_TRIGGER_MAX_INDEX (else CBM_ERR_CAPACITY); no atomics, the output is unique.  Scratch is allocated and freed
 * on `stream` (cudaMallocAsync).  An event built from more than max_hits_per_layer hits in a layer is rejected by the
 * selection like any other such event (CBM_ERR_RANGE). */
int cbm_trigger_build_events_device(cbm_trigger_t* h, uint64_t n_records, const int32_t* d_t, uint32_t t_gap,
                                    uint32_t* d_ev_off, uint32_t* n_events, void* stream);

/* The paper's own selection, literally (section 3.2), on caller-owned DEVICE
 * arrays (layout and stream as cbm_trigger_run_device; geometry = the handle's layer_z):
 *   1. all triplets of the trigger station, one hit from each layer
 *   2. least-squares line through the event vertex (0,0) in x-z and in y-z (x = m0 z, y = m1 z), mean square
 *      deviation per degree of freedom <= thr_x (0.03) in x-z and <= thr_y (0.025) in y-z
 *   3. d_accept[e] = d_n_passing[e] >= min_triplets (2)
 * evaluated exactly: with Svz = sum v_i z_i, Szz = sum z_i^2, Svv = sum v_i^2 over the three hits,
 *   den * (Szz*Svv - Svz^2) <= num * 10^6 * ndf * Szz      (thr = num/den cm^2; 10-um units; 128-bit integers),
 * exact for any int32 x, y.  d_n_passing[n_events] uint32 = min(2^32-1, passing triplets); d_accept uint8.
 * An event with malformed offsets has d_n_passing = 0 and d_accept = 0 (also with min_triplets = 0).  Asynchronous. */
typedef struct {
  uint32_t struct_size;            /* = sizeof(cbm_trigger_msd_params_t) */
  uint32_t station;                /* the trigger station, 0..S-1; 0xFFFFFFFF = the last one */
  uint32_t thr_x_num, thr_x_den;   /* MSD_xz threshold in cm^2 (0.03 = 3/100); den 1..4096, num <= 2^20 */
  uint32_t thr_y_num, thr_y_den;   /* MSD_yz threshold (0.025 = 25/1000) */
  uint32_t ndf;                    /* degrees of freedom, 1..16 (2: three hits, one fitted slope) */
  uint32_t min_triplets;           /* 2 */
} cbm_trigger_msd_params_t;
int cbm_trigger_msd_device(cbm_trigger_t* h, const cbm_trigger_msd_params_t* params, uint32_t n_events, uint64_t n_hits,
                           const int32_t* d_x, const int32_t* d_y, const uint32_t* d_off, uint32_t* d_n_passing,
                           uint8_t* d_accept, void* stream);

/* Device-resident entry point (PyTorch or any other owner of device memory and streams supplies both):
 * runs a3-a8 on caller-owned DEVICE arrays on the caller's stream (`stream` is a cudaStream_t passed as void*;
 * NULL = the legacy default stream).  d_x, d_y: n_hits int32 each, 16-byte aligned, readable up to the next
 * multiple of 4 elements (over-read by the 128-bit staging copies; contents ignored).  d_off: n_events*L+1
 * uint32.  Outputs: d_n_triplets[n_events*S] uint32, d_n_candidates[n_events] uint32, d_accept[n_events] uint8.
 * Asynchronous; the handle's scheduler scratch is reused, so calls on one handle must be stream-ordered.
 * Requires n_events <= max_events.  Structural errors are reported by cbm_trigger_device_status(). */
int cbm_trigger_run_device(cbm_trigger_t* h, uint32_t n_events, uint64_t n_hits, const int32_t* d_x,
                           const int32_t* d_y, const uint32_t* d_off, uint32_t* d_n_triplets,
                           uint32_t* d_n_candidates, uint8_t* d_accept, void* stream);

/* Synchronises `stream` and fills *stats (HOST) for the last cbm_trigger_run_device call.  Returns
 * CBM_ERR_RANGE if that run rejected events, CBM_OK otherwise. */
int cbm_trigger_device_status(cbm_trigger_t* h, void* stream, cbm_trigger_stats_t* stats);

/* CBM_FLAG_PROFILE only: synchronises `stream`, then writes the device time in ms of every kernel of the last
 * min(n_last, CBM_TRIGGER_PROFILE_RING, calls so far) cbm_trigger_run_device calls, oldest first, to the HOST
 * array kernel_ms[call*CBM_TRIGGER_N_KERNELS + kernel] (CUDA events recorded on the launching stream).
 * Returns the number of calls written (>= 0) or a negative error code. */
int cbm_trigger_device_kernel_times(cbm_trigger_t* h, void* stream, uint32_t n_last, float* kernel_ms);

/* Measurement utility (the integer-pipe denominators of the roofline are measured on the box,
 * not taken from a data sheet): runs four micro-benchmarks on the handle's device (8 independent dependency
 * chains per thread, 8 CTAs of 256 threads per SM) and blocks until they are done.  Lane operations per second
 * of the INT32 ALU pipe (IADD3 + LOP3) and of the FMA pipe (IMAD); exact window evaluations per second (one
 * evaluation = the int64 test in x and in y, as the kernels compile it; PAPER.md:75-76 is the test it stands
 * for); packed key tests per second.  out: HOST, struct_size set by the caller. */
typedef struct {
  uint32_t struct_size;  /* = sizeof(cbm_trigger_ubench_t) */
  uint32_t n_sm;
  double alu_lane_ops_per_s;
  double imad_lane_ops_per_s;
  double window_evals_per_s;
  double packed_tests_per_s;
} cbm_trigger_ubench_t;
int cbm_trigger_ubench(cbm_trigger_t* h, cbm_trigger_ubench_t* out);

/* Statistics of the last completed run of `slot` (call after fetch_results).  stats: HOST. */
int cbm_trigger_get_stats(cbm_trigger_t* h, uint32_t slot, cbm_trigger_stats_t* stats);

/* Handle-owned, NUL-terminated message of the last failing call ("" if none).  With h == NULL: the message of
 * the last failing cbm_trigger_create or cbm_trigger_select_noalloc on this thread. */
const char* cbm_trigger_last_error(const cbm_trigger_t* h);

/* "cbm-trigger <version> sm_100a" */
const char* cbm_trigger_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CBM_TRIGGER_H */
