/* tt.h -- C ABI of the B200 tower-trigger library (libtt.so).
 *
 * The hot path of the online muon trigger of "Parallel Neutrino Triggers using GPUs for an
 * Underwater Telescope" (arxiv 1411.3968; citations are lines of PAPER.md), as scoped by
 * BASELINE.json:north_star:
 *
 *   tt_sort_slice      PAPER.md:51-53 (sect. 4.2 "First we sort the hits in time"; the per-PMT streams
 *                      are already time-ordered)            -- stable time sort
 *   tt_trigger_slice   PAPER.md:27-29 (sect. 3: charge over threshold, time-space correlation within
 *                      3 us), PAPER.md:61-64 (coincidences, QTRIG)       -- L1, L2, seed list
 *   tt_extract_events  PAPER.md:23 ("a 6 us time window ... centered at the time of the trigger seed"),
 *                      PAPER.md:67 ("all hits within +-3 us are tagged") -- event-window merge, tagging
 *   tt_l0_ntw          PAPER.md:59, 67, 73 (N7TW1000 / N7TW500, the paper's level-0 trigger) -- N hits in TW
 *   tt_l0_dntw         PAPER.md:60 (DN7TW1000: N hits from different PMTs in TW)   -- distinct-PMT level-0 trigger
 *   tt_pair_seeds      PAPER.md:61-63 (SC, FC, AFC coincidences)          -- the paper's pair seeds
 *   tt_l0_combine      PAPER.md:65, 73 (N7TW with [SC and AFC] or [FC and AFC]) -- the paper's combined trigger
 *   tt_prepare_slice   PAPER.md:41-47 (raw hits -> fixed-size records, slices packed into one buffer) -- preparation
 *   tt_sort_trigger_slice  tt_sort_slice + tt_trigger_slice as one call, L1 fused into the last merge level
 *
 * Conventions
 *   d_*   device pointers (caller-owned; the library never allocates in the three hot calls)
 *   h_*   host pointers; `p`, `g`, `ws_bytes` are host pointers too
 *   All hot calls are asynchronous: they enqueue kernels on `stream` (a cudaStream_t passed as
 *   void*) and return.  The return value covers argument errors only (TT_OK / TT_E_*).
 *   The library keeps no state between calls apart from per-device one-time kernel set-up and a per-host-thread copy
 *   of the last merge plan (both invisible in the results); calls from several host threads and on several devices
 *   are allowed.
 *   Data-dependent conditions are OR-ed into *d_status (device int32, zeroed by the caller or by
 *   a previous call's owner), to be read after synchronising: TT_S_* bits.
 *   Workspace: call with d_ws == NULL to get the required size in *ws_bytes (nothing is enqueued);
 *   otherwise *ws_bytes must be >= that size.  d_ws must be 256-byte aligned.
 *   Indices are uint32: n < 2^32 - 2^20.
 *   Segments: d_seg_offsets[n_seg+1] (device) splits the hit array into independent slices
 *   (no sort movement, coincidence or event crosses a segment).  h_seg_offsets is the same array
 *   on the host (needed to size launches); both must agree.
 */
#ifndef TT_H_
#define TT_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Fixed-size hit record ("a fixed size structure": charge, time, DU identification);
 * 16 bytes, 16-byte aligned.  t_ps: picoseconds, any int64.  floor: global floor id (tower*floors+f).
 * charge: 0.01 p.e. units.  pad: carried through unchanged. */
typedef struct {
    int64_t t_ps;
    uint16_t pmt_id, floor, charge, pad;
} tt_hit;

/* Trigger parameters (BASELINE.json configs[0]); 40 bytes, no implicit padding. */
typedef struct {
    int64_t lc_window_ps;     /* L1 same-floor coincidence window, inclusive (20000)              */
    int64_t l2_window_ps;     /* W: an L2 edge needs |dt| <= min(dtmax, W), inclusive (3000000)    */
    int64_t event_half_ps;    /* H: event window is [t_seed - H, t_seed + H] (3000000)             */
    uint32_t l2_multiplicity; /* N >= 1, counts the hit itself; N <= TT_MAX_MULTIPLICITY           */
    uint32_t l2_mode;         /* 0 = clique ("N L1 hits pairwise causal"), 1 = star                */
    uint32_t q_thresh;        /* Q bit <=> charge >= q_thresh (0.01 p.e.; PAPER.md:64 QTRIG)       */
    uint32_t l1_capacity;     /* 0: the L1 list may hold every hit (workspace ~69 B per hit).  Else the most L1
                                 hits per call the trigger workspace is sized for (~69 B each; a detector has
                                 2-8 % L1 hits): with more, TT_S_L1_OVERFLOW is set, the L1 flags of all hits
                                 are still exact, and L2 / seeds see the first l1_capacity L1 hits of the sorted array  */
} tt_params;

/* One merged event window; 32 bytes.  Times are unclipped; [hit_begin, hit_end) indexes the sorted
 * hit array, [seed_begin, seed_begin + n_seeds) indexes the seed list. */
typedef struct {
    int64_t t_start, t_end;
    uint32_t hit_begin, hit_end, seed_begin, n_seeds;
} tt_event;

/* per-hit flag byte */
enum { TT_Q = 1, TT_LC = 2, TT_L1 = 4, TT_L2STAR = 8, TT_L2 = 16, TT_INEVT = 32 };
/* return codes */
enum { TT_OK = 0, TT_E_INVAL = -1, TT_E_CUDA = -2, TT_E_WORKSPACE = -3,
       TT_E_LIMIT = -4 /* tt_extract_events_noalloc: the request needs more than TT_NOALLOC_WS_BYTES of scratch */ };
/* *d_status bits */
enum {
    TT_S_OK = 0,
    TT_S_SEED_OVERFLOW = 1,  /* n_seeds > seed_cap: *d_n_seeds is the true count, first seed_cap valid */
    TT_S_EVENT_OVERFLOW = 2, /* likewise for events                                                   */
    TT_S_RUN_UNSORTED = 4,   /* a run given by d_run_offsets is not non-decreasing: output unspecified */
    TT_S_BAD_PMT = 8,        /* an L1 hit has pmt_id >= n_pmt (it has no L2 edges)                     */
    TT_S_L1_OVERFLOW = 64,   /* tt_l1_export: more L1 hits than l1_cap (*d_n_l1 is the true count, first l1_cap valid);
                                tt_trigger_slice / tt_sort_trigger_slice: more L1 hits than tt_params.l1_capacity      */
    TT_S_RAW_TRUNCATED = 32, /* tt_prepare_slice: a waveform reaches behind the sample section (missing samples = 0) */
    TT_S_DENSITY = 16        /* an L1 hit has more than TT_MAX_NEIGHBOURS L1 hits of its segment within
                                +-min(W, largest table entry) of it: its L2STAR bit is exact, and its
                                clique-mode L2 bit is SET FROM the L2STAR bit (fail open: a superset of
                                the exact answer, the same on every run; the hit stays in the data)  */
};
#define TT_MAX_MULTIPLICITY 16
#define TT_MAX_NEIGHBOURS 2048
#define TT_MAX_L0_MULTIPLICITY 256
#define TT_MAX_DN_MULTIPLICITY 16
/* per-hit byte of tt_l0_ntw */
enum { TT_L0_START = 1, TT_L0_MEMBER = 2 };
/* per-hit byte of tt_pair_seeds (SC, FC, AFC) and of tt_l0_combine (CAND_A, CAND_B) */
enum { TT_P_SC = 1, TT_P_FC = 2, TT_P_AFC = 4, TT_P_CAND_A = 8, TT_P_CAND_B = 16 };

/* Causality table dtmax[pmt_a][pmt_b] in integer ps (BASELINE.json configs[0]: d_ij*n/c + 20 ns,
 * precomputed by the caller), block-sparse by tower pair:
 *   dtmax(a, b) = h_blocks[h_pair_block[ta*n_tower + tb]][a % ppt][b % ppt],  ta = a / ppt,
 * -1 (block id or entry) = the pair is never an edge.  One tower: n_tower = 1, h_pair_block = {0}.
 * The table is copied to the device; tt_geometry_destroy frees it.  Returns TT_E_INVAL for a
 * non-symmetric table, a block id out of range, or n_pmt != n_tower * pmts_per_tower. */
typedef struct tt_geometry tt_geometry;
int tt_geometry_create(tt_geometry** g, uint32_t n_pmt, uint32_t n_tower, uint32_t pmts_per_tower,
                       const int32_t* h_pair_block, const int32_t* h_blocks, uint32_t n_blocks);
int tt_geometry_destroy(tt_geometry* g);

/* Stable ascending sort of d_in[n] by t_ps inside each segment (ties keep input order) into
 * d_out[n] (a pure permutation of whole 16-byte records; d_out must not alias d_in).
 * d_perm (nullable): d_perm[k] = input index of d_out[k].
 * d_run_offsets[n_runs+1] (nullable, with its host copy h_run_offsets): consecutive, already
 * non-decreasing runs covering [0, n) that never straddle a segment (the per-PMT streams).  Given,
 * the library merges the runs; NULL, it radix-sorts arbitrary input.  A run that is not sorted sets
 * TT_S_RUN_UNSORTED. */
int tt_sort_slice(const tt_hit* d_in, tt_hit* d_out, uint32_t* d_perm, uint32_t n,
                  const uint32_t* d_seg_offsets, const uint32_t* h_seg_offsets, uint32_t n_seg,
                  const uint32_t* d_run_offsets, const uint32_t* h_run_offsets, uint32_t n_runs,
                  void* d_ws, size_t* ws_bytes, int32_t* d_status, void* stream);

/* L1 (Q | same-floor coincidence on another PMT within lc_window), L2 (clique or star over the
 * causality table within l2_window) and the ascending seed list on time-sorted hits.
 * d_flags[n] is overwritten (TT_Q..TT_L2 bits).  d_seeds[seed_cap] receives the sorted-array
 * indices of the L2 hits, *d_n_seeds the true count. */
int tt_trigger_slice(const tt_hit* d_sorted, uint32_t n, const uint32_t* d_seg_offsets,
                     const uint32_t* h_seg_offsets, uint32_t n_seg, const tt_geometry* g,
                     const tt_params* p, uint8_t* d_flags, uint32_t* d_seeds, uint32_t seed_cap,
                     uint32_t* d_n_seeds, void* d_ws, size_t* ws_bytes, int32_t* d_status, void* stream);

/* tt_sort_slice followed by tt_trigger_slice as ONE call (last bullet):
 * the same arguments, the same outputs byte for byte (d_out, d_perm, d_flags, d_seeds, *d_n_seeds, status bits).
 * With runs given, the L1 step (Q | same-floor coincidence) is evaluated by the last merge level on its time tile
 * while the sorted tile is in shared memory, so the sorted array is not read a second time for it; the hits within
 * lc_window of a tile edge are finished by exact scans afterwards (the paper's "edge" rule between sub-slices,
 * PAPER.md:47).  Without runs it is the two calls back to back.  Workspace = both calls' workspaces; same alignment
 * and error rules as the two calls. */
int tt_sort_trigger_slice(const tt_hit* d_in, tt_hit* d_out, uint32_t* d_perm, uint32_t n,
                          const uint32_t* d_seg_offsets, const uint32_t* h_seg_offsets, uint32_t n_seg,
                          const uint32_t* d_run_offsets, const uint32_t* h_run_offsets, uint32_t n_runs,
                          const tt_geometry* g, const tt_params* p, uint8_t* d_flags, uint32_t* d_seeds,
                          uint32_t seed_cap, uint32_t* d_n_seeds, void* d_ws, size_t* ws_bytes, int32_t* d_status,
                          void* stream);

/* Merge the closed windows [t-H, t+H] of consecutive seeds (merge <=> gap <= 2H, never across a
 * segment) into d_events[event_cap]; *d_n_events = true count.  The seed list is read from the
 * device (d_seeds, *d_n_seeds as written by tt_trigger_slice; at most seed_cap entries are used).
 * d_flags (nullable): TT_INEVT is OR-ed into the flags of every hit inside an event.
 * d_gather (nullable, room for n records): the hits of all events, concatenated in order;
 * *d_n_gathered (nullable) = their number. */
int tt_extract_events(const tt_hit* d_sorted, uint32_t n, const uint32_t* d_seg_offsets,
                      const uint32_t* h_seg_offsets, uint32_t n_seg, const uint32_t* d_seeds,
                      const uint32_t* d_n_seeds, uint32_t seed_cap, const tt_params* p,
                      tt_event* d_events, uint32_t event_cap, uint32_t* d_n_events, uint8_t* d_flags,
                      tt_hit* d_gather, uint32_t* d_n_gathered, void* d_ws, size_t* ws_bytes,
                      int32_t* d_status, void* stream);

/* tt_extract_events for callers that cannot allocate device memory (code under CUDA-graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): the same operation, the same arguments minus the
 * workspace pair, the same outputs byte for byte -- the scratch the kernels need (per-block counts, the head flag of
 * every seed, the gather offset of every event: 4 * event_cap + seed_cap + ~5 KB) lives in a static device array of
 * TT_NOALLOC_WS_BYTES inside the library, which every GPU that loads the library holds until the process exits.
 *   - seed_cap / event_cap whose scratch does not fit return TT_E_LIMIT and launch nothing (e.g. event_cap = 2^18
 *     with seed_cap = 2^21 fits; cfg4 has 1.18 M seeds and 405 events per slice);
 *   - the call makes no cudaMalloc / cudaFree and calls no allocating library routine; the first call on a device
 *     resolves the array's device address (cudaGetSymbolAddress, once per device, that device current), so make that
 *     first call outside stream capture;
 *   - ALL calls on a device share the one array, which keeps the last call's contents (nothing in it has to start at
 *     zero: every word a kernel reads was written earlier in the same call): two calls that overlap on the GPU
 *     (different streams, no dependency between them) race on it.  Calls on one stream are ordered and safe. */
#define TT_NOALLOC_WS_BYTES (4u << 20)
int tt_extract_events_noalloc(const tt_hit* d_sorted, uint32_t n, const uint32_t* d_seg_offsets,
                              const uint32_t* h_seg_offsets, uint32_t n_seg, const uint32_t* d_seeds,
                              const uint32_t* d_n_seeds, uint32_t seed_cap, const tt_params* p,
                              tt_event* d_events, uint32_t event_cap, uint32_t* d_n_events, uint8_t* d_flags,
                              tt_hit* d_gather, uint32_t* d_n_gathered, int32_t* d_status, void* stream);

/* Level-0 N-in-TW trigger on time-sorted hits: "N7TW1000: looking for 7 hits
 * in TW = 1000 ns: hit[i].time-hit[i+7].time< TW", PAPER.md:73 (N7TW500 for the 84-PMT tower), PAPER.md:67 (applied
 * first, "as level 0 trigger").  Reading R14 / R20 of DESIGN.md: inside each segment, window start k fires <=> hit
 * k + N - 1 exists in k's segment and t[k+N-1] - t[k] < window_ps (strict, as printed; window_ps <= 0 never fires).
 * d_l0[n] (device, overwritten): TT_L0_START = the hit is a firing window start, TT_L0_MEMBER = the hit is one of the
 * N hits k..k+N-1 of some firing window.  d_n_start (device, nullable): number of firing starts (zeroed by the call).
 * d_sorted must be time-sorted inside each segment (the output of tt_sort_slice); unsorted input gives unspecified
 * bits, never an out-of-bounds access.  multiplicity N in [1, TT_MAX_L0_MULTIPLICITY], else TT_E_INVAL.  No
 * workspace, no status bits; asynchronous on `stream`. */
int tt_l0_ntw(const tt_hit* d_sorted, uint32_t n, const uint32_t* d_seg_offsets, uint32_t n_seg,
              uint32_t multiplicity, int64_t window_ps, uint8_t* d_l0, uint32_t* d_n_start, void* stream);

/* Distinct-PMT level-0 trigger DNnTW (rest of SURVEY.md 8(f) NEXT-1): "DN7TW1000: looking for 7 hits
 * from different PMTs within TW = 1000 ns".  Reading R23 of DESIGN.md: inside each segment, window start k fires <=> the
 * hits j >= k with t_j - t_k < window_ps (strict) carry at least N different pmt_id values; its members are the hits
 * k..e_k, e_k = the first hit at which the N-th different PMT appears (with all PMTs different: tt_l0_ntw's window).
 * d_l0[n] (device; zeroed, then written, by the call): TT_L0_START | TT_L0_MEMBER as for tt_l0_ntw.  d_n_start
 * (device, nullable): number of firing starts.  multiplicity N in [1, TT_MAX_DN_MULTIPLICITY], else TT_E_INVAL.
 * Exact for any hit density (windows longer than the staged tile are finished from global memory).  No workspace, no
 * status bits; asynchronous on `stream`. */
int tt_l0_dntw(const tt_hit* d_sorted, uint32_t n, const uint32_t* d_seg_offsets, uint32_t n_seg,
               uint32_t multiplicity, int64_t window_ps, uint8_t* d_l0, uint32_t* d_n_start, void* stream);

/* The paper's pair-coincidence seeds on time-sorted hits, PAPER.md:61-63:
 *   TT_P_SC   "two hits occurred in two adjacent PMTs within 20 ns": same tower (pmt_id / pmts_per_tower) and
 *             d_adj[(pmt_a % ppt) * ppt + pmt_b % ppt] != 0, |dt| <= sc_window_ps
 *   TT_P_FC   "two PMTs in the same floor within 100 ns": equal `floor` fields, |dt| <= fc_window_ps
 *   TT_P_AFC  "two PMTs located at two consecutive floors within 250 ns": same tower, `floor` fields differing by
 *             exactly 1, |dt| <= afc_window_ps
 * A pair is two hits of one segment on two DIFFERENT PMTs; windows are inclusive (readings R4, R5, R21).
 * d_adj: device, uint8[ppt * ppt], symmetric, the caller's "adjacent PMTs" relation over one tower's PMTs.
 * d_bits[n] (device, overwritten): OR of the rule bits over all partners of the hit.  Windows must be >= 0 and
 * pmts_per_tower in [1, 65535], else TT_E_INVAL.  No workspace, no status bits; asynchronous on `stream`. */
int tt_pair_seeds(const tt_hit* d_sorted, uint32_t n, const uint32_t* d_seg_offsets, uint32_t n_seg,
                  const uint8_t* d_adj, uint32_t pmts_per_tower, int64_t sc_window_ps, int64_t fc_window_ps,
                  int64_t afc_window_ps, uint8_t* d_bits, void* stream);

/* The paper's combined trigger, PAPER.md:65, 73 ("applying N7TW1000, and if it is satisfied, we apply [SC and AFC]
 * or [FC and AFC] ... used to tag the muon track candidate"; reading R22): for every firing level-0 window
 * start k (d_l0[k] & TT_L0_START, as written by tt_l0_ntw with the same multiplicity N), the pair bits of its N hits
 * k..k+N-1 are OR-ed; d_cand[k] gets TT_P_CAND_A when SC and AFC both occur among them, TT_P_CAND_B when FC and AFC
 * both occur.  Every other byte of d_cand[n] is 0.  d_n_cand (device, nullable, uint32[2], zeroed by the call):
 * number of CAND_A and of CAND_B starts. */
int tt_l0_combine(const uint8_t* d_l0, const uint8_t* d_pair_bits, uint32_t n, uint32_t multiplicity,
                  uint8_t* d_cand, uint32_t* d_n_cand, void* stream);

/* The paper's preparation step on the GPU ("the raw hits are converted to a fixed
 * size structure", PAPER.md:45 five 200 ms slices packed into one buffer at offsets: 200-300 ms of CPU
 * time per second of data in the paper).  The paper does not give its raw format; this build's (reading R24):
 *   d_raw[n_raw]     16-byte headers in ARRIVAL order: every PMT's hits time-ordered, the PMTs interleaved
 *   d_samples[...]   the sampled charge waveforms of all hits, concatenated in the same order, uint16 each; hit k owns
 *                    n_samples_k samples starting at the sum of the sample counts before it (< 2^32 in total)
 *   d_slice_offsets  [n_slices + 1] (device; h_slice_offsets = the same on the host) cut d_raw into 200 ms slices
 * Output: d_out[n_raw] fixed-size records {t_ps, pmt_id, floor, charge = min(65535, sum of the samples), pad} ordered
 * slice-major, then PMT-major, arrival order kept inside a (slice, PMT) run -- the concatenated, individually
 * time-ordered runs tt_sort_slice takes -- and d_run_offsets[n_slices * n_pmt + 1] (device), their offsets.  (The host
 * copy tt_sort_slice also wants is a 4-byte-per-run read-back by the caller.)  n_raw > out_cap (the buffer the caller
 * sized: for 5 x the nominal rate) returns TT_E_INVAL.  Status bits: TT_S_BAD_PMT (pmt_id >= n_pmt: the
 * hit is filed under the last PMT of its slice, record unchanged), TT_S_RAW_TRUNCATED.  Asynchronous on `stream`. */
typedef struct {
    int64_t t_ps;
    uint16_t pmt_id, floor, n_samples, pad;
} tt_raw_hit;
int tt_prepare_slice(const tt_raw_hit* d_raw, const uint16_t* d_samples, uint32_t n_raw, uint32_t n_samples_total,
                     const uint32_t* d_slice_offsets, const uint32_t* h_slice_offsets, uint32_t n_slices,
                     uint32_t n_pmt, tt_hit* d_out, uint32_t out_cap, uint32_t* d_run_offsets, void* d_ws,
                     size_t* ws_bytes, int32_t* d_status, void* stream);

/* ---- A multi-tower detector sharded BY TOWER over several GPUs, with one exchange (
 * PAPER.md:81, sect. 5: "each TGPU finds the trigger seeds of its tower and sends them to a TCPU ... gets candidate
 * times back").  L1 is local to a floor, hence to a tower; only L2 and the event windows look across towers.  Per rank
 * (a contiguous range of towers; pmt ids and floor ids stay GLOBAL):
 *   tt_sort_l1_slice   its hits -> time-sorted + Q / LC / L1 flag bytes (tt_sort_trigger_slice without L2 / seeds;
 *                      runs required);
 *   tt_l1_export       its L1 hits, in sorted order, as 16-byte records {t_ps, idx = sorted index, pmt_id, src = rank};
 *   -- the ranks all-gather their records (NCCL; ~2 % of the hits) and concatenate them in rank order --
 *   tt_sort_slice      on the concatenation (one run per rank; the record starts with the time, like a hit) merges it;
 *   tt_l2_merged       L2STAR / L2 of every record of the merged list (the L2 kernels of tt_trigger_slice; same
 *                      geometry, same status bits) into d_bits[m], and the positions of the L2 records -- the GLOBAL
 *                      seed list, identical on every rank -- into d_seeds;
 *   tt_extract_events  on (merged list as hits, d_seeds) gives the global event windows (t_start, t_end, seed_begin,
 *                      n_seeds as on one GPU; hit_begin / hit_end index the merged list);
 *   tt_l2_apply        writes the L2STAR / L2 bits of the rank's own records into its flag bytes and its own seeds
 *                      (ascending sorted indices) into d_seeds;
 *   tt_tag_windows     ORs TT_INEVT into the flags of the rank's hits inside any of the global windows.
 * Flags, seeds (per rank) and window times then equal, hit for hit, what one GPU computes on the whole detector.
 * Workspace / status / stream conventions as above. */
typedef struct {
    int64_t t_ps;
    uint32_t idx;
    uint16_t pmt_id, src;
} tt_l1hit;
int tt_sort_l1_slice(const tt_hit* d_in, tt_hit* d_out, uint32_t* d_perm, uint32_t n, const uint32_t* d_seg_offsets,
                     const uint32_t* h_seg_offsets, uint32_t n_seg, const uint32_t* d_run_offsets,
                     const uint32_t* h_run_offsets, uint32_t n_runs, const tt_params* p, uint8_t* d_flags, void* d_ws,
                     size_t* ws_bytes, int32_t* d_status, void* stream);
int tt_l1_export(const tt_hit* d_sorted, uint32_t n, const uint8_t* d_flags, uint32_t src, tt_l1hit* d_l1, uint32_t l1_cap,
                 uint32_t* d_n_l1, void* d_ws, size_t* ws_bytes, int32_t* d_status, void* stream);
int tt_l2_merged(const tt_l1hit* d_l1, uint32_t m, const tt_geometry* g, const tt_params* p, uint8_t* d_bits,
                 uint32_t* d_seeds, uint32_t seed_cap, uint32_t* d_n_seeds, void* d_ws, size_t* ws_bytes,
                 int32_t* d_status, void* stream);
int tt_l2_apply(const tt_l1hit* d_l1, const uint8_t* d_bits, uint32_t m, uint32_t src, uint8_t* d_flags, uint32_t n,
                uint32_t* d_seeds, uint32_t seed_cap, uint32_t* d_n_seeds, void* d_ws, size_t* ws_bytes,
                int32_t* d_status, void* stream);
int tt_tag_windows(const tt_hit* d_sorted, uint32_t n, const tt_event* d_events, const uint32_t* d_n_events,
                   uint32_t event_cap, const tt_params* p, uint8_t* d_flags, void* stream);

/* Whole-slice convenience with HOST buffers (end-to-end use and timing; not a hot call).
 * tt_host_ctx_create allocates, once, device buffers and workspaces for slices of up to max_n hits,
 * max_seg segments and max_runs runs, and an internal stream; tt_host_ctx_destroy frees them.
 * tt_process_host copies the hits and offsets to the device (h_in pinned or pageable), runs
 * tt_sort_trigger_slice -> tt_extract_events (with INEVT tagging), copies back the
 * sorted hits (h_sorted nullable), the flags (h_flags nullable), the first min(n_seeds, seed_cap)
 * seeds and min(n_events, event_cap) events, and synchronises.
 * h_counts[3] = {n_seeds, n_events, status}.  h_run_offsets NULL = unsorted input. */
typedef struct tt_host_ctx tt_host_ctx;
int tt_host_ctx_create(tt_host_ctx** c, uint32_t max_n, uint32_t max_seg, uint32_t max_runs, uint32_t seed_cap,
                       uint32_t event_cap);
int tt_host_ctx_destroy(tt_host_ctx* c);
/* The same, two slices deep, for slices that arrive back to back: tt_host_submit enqueues the upload of
 * a slice, its compute and the read-back of its results on three streams and returns at once; the upload of the next
 * slice then overlaps this slice's compute and the previous slice's read-back.  tt_host_wait blocks until the OLDEST
 * submitted slice is complete (its h_* buffers and h_counts are then valid).  At most two slices may be in flight
 * (a third tt_host_submit returns TT_E_INVAL); the host buffers of a slice must stay untouched until its wait returns.
 * tt_process_host = tt_host_submit + tt_host_wait. */
int tt_host_submit(tt_host_ctx* c, const tt_hit* h_in, tt_hit* h_sorted, uint8_t* h_flags, uint32_t n,
                   const uint32_t* h_seg_offsets, uint32_t n_seg, const uint32_t* h_run_offsets, uint32_t n_runs,
                   const tt_geometry* g, const tt_params* p, uint32_t* h_seeds, tt_event* h_events,
                   uint32_t* h_counts);
int tt_host_wait(tt_host_ctx* c);
int tt_process_host(tt_host_ctx* c, const tt_hit* h_in, tt_hit* h_sorted, uint8_t* h_flags, uint32_t n,
                    const uint32_t* h_seg_offsets, uint32_t n_seg, const uint32_t* h_run_offsets,
                    uint32_t n_runs, const tt_geometry* g, const tt_params* p, uint32_t* h_seeds,
                    tt_event* h_events, uint32_t* h_counts);

/* Instrumentation (not on the data path).  tt_launch_count: kernels launched by this library in
 * this process so far.  tt_prof_enable(1) makes every stage boundary inside the hot calls record a
 * CUDA event on the caller's stream; after synchronising, tt_prof_read writes one line per stage,
 * "name total_ms count", into buf (returns bytes written, < 0 on error); tt_prof_enable(0) stops. */
uint64_t tt_launch_count(void);
int tt_prof_enable(int on);
int tt_prof_read(char* buf, size_t cap);

/* Library version / build string (static storage). */
const char* tt_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TT_H_ */
