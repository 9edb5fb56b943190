// oracle/tt_oracle.cpp -- TEST INFRASTRUCTURE, not product code.
//
// Plain, slow, single-threaded CPU definition of the hot path of the online muon trigger of
// "Parallel Neutrino Triggers using GPUs for an Underwater Telescope" (arxiv 1411.3968),
// as scoped by BASELINE.json:north_star.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may load this library.  It shares no code, headers,
// tables or helpers with paper_1411_3968_b200/csrc (the CUDA path); the record layouts below
// are re-declared here on purpose.
//
// What each function follows:
//   oracle_sort     PAPER.md:51-53 (sect. 4.2 "First we sort the hits in time"); north_star "put
//                   them in global timestamp order (a merge of the per-PMT time-ordered streams)".
//                   The plain definition: std::stable_sort by t_ps inside each segment
//                   (reading R2: ties keep input order).
//   oracle_trigger  PAPER.md:27-29 (sect. 3: charge over threshold; time-space correlation within
//                   3 us), PAPER.md:61-64 (SC/FC coincidences, QTRIG) with the windows and the
//                   pairwise L2 condition of north_star / BASELINE.json configs[0].
//   oracle_events   PAPER.md:23 ("a 6 us time window ... centered at the time of the trigger
//                   seed"), PAPER.md:67 ("all hits within +-3 us are tagged").
//   oracle_pair_seeds  PAPER.md:61-63: SC ("two hits occurred in two adjacent PMTs within 20 ns"), FC ("two PMTs in the
//                   same floor within 100 ns"), AFC ("two PMTs located at two consecutive floors within 250 ns").
//   oracle_l0_combine  PAPER.md:65, 73: "applying N7TW1000, and if it is satisfied, we apply [SC and AFC] or [FC and
//                   AFC]" (reading R22: evaluated over the N hits of each firing level-0 window).
//   oracle_l0_dntw  PAPER.md:60 ("DN7TW1000: looking for 7 hits from different PMTs within TW = 1000 ns"); DESIGN.md
//                   reading R23.
//   oracle_l0_ntw   PAPER.md:59 ("N7TW1000: looking for 7 hits in TW = 1000 ns:
//                   hit[i].time-hit[i+7].time< TW"), PAPER.md:73 (N7TW500 for the 84-PMT tower)
//                   (used first, "as level 0 trigger").  DESIGN.md reading R14: the printed formula has the
//                   sign reversed and 7 hits span i..i+6, so the test is t[k+N-1] - t[k] < TW, strict as printed.
//
//   oracle_prepare  PAPER.md:41 ("the raw hits are converted to a fixed size structure": charge, time, DU id),
//                   PAPER.md:45 (five 200 ms slices packed into one buffer at offsets), PAPER.md:23 (each PMT's
//                   stream is time-ordered, the merged stream is not PMT-major).  DESIGN.md reading R24 (the raw
//                   format is this build's: the paper gives none).
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): brute-force pair / subset enumeration written
// separately in oracle/brute.py, numpy stable argsort, Poisson closed forms, N-in-TW special
// case, interval-union brute force, hand-written boundary cases.  No function
// here is "parity unpinned".
#include <algorithm>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

struct Hit {
    int64_t t_ps;
    uint16_t pmt_id, floor, charge, pad;
};
static_assert(sizeof(Hit) == 16, "hit record is 16 bytes");

struct Params {
    int64_t lc_window_ps;
    int64_t l2_window_ps;
    int64_t event_half_ps;
    uint32_t l2_multiplicity;
    uint32_t l2_mode;  // 0 clique, 1 star
    uint32_t q_thresh;
    uint32_t reserved;
};
static_assert(sizeof(Params) == 40, "params layout");

struct Event {
    int64_t t_start, t_end;
    uint32_t hit_begin, hit_end, seed_begin, n_seeds;
};
static_assert(sizeof(Event) == 32, "event record is 32 bytes");

enum : uint8_t { F_Q = 1, F_LC = 2, F_L1 = 4, F_L2STAR = 8, F_L2 = 16, F_INEVT = 32 };
enum : int32_t { S_BAD_PMT = 8 };

struct Geo {
    uint32_t n_pmt, n_tower, ppt;
    const int32_t* pair_block;  // [n_tower*n_tower], -1 = unconnected
    const int32_t* blocks;      // [n_blocks][ppt][ppt] ps
};

// dtmax(pmt_a, pmt_b): the integer causality table; -1 = never an edge.
int64_t dtmax(const Geo& g, uint32_t a, uint32_t b) {
    if (a >= g.n_pmt || b >= g.n_pmt) return -1;
    const uint32_t ta = a / g.ppt, tb = b / g.ppt;
    const int32_t blk = g.pair_block[(size_t)ta * g.n_tower + tb];
    if (blk < 0) return -1;
    return g.blocks[((size_t)blk * g.ppt + (a % g.ppt)) * g.ppt + (b % g.ppt)];
}

// Exact t_hi - t_lo for t_hi >= t_lo (hits are time-sorted where this is used).  DESIGN.md reading R1: timestamps are
// "any int64", so a span can reach 2^64 - 1 and does not fit int64; it always fits uint64.
uint64_t span(int64_t t_hi, int64_t t_lo) { return (uint64_t)t_hi - (uint64_t)t_lo; }

// Is there a subset of `need` members of cand[from..], pairwise adjacent?  Plain recursion.
bool has_clique(const std::vector<std::vector<uint8_t>>& adj, const std::vector<int>& cand, int need) {
    if (need == 0) return true;
    if ((int)cand.size() < need) return false;
    for (size_t k = 0; k < cand.size(); ++k) {
        const int v = cand[k];
        std::vector<int> rest;
        for (size_t m = k + 1; m < cand.size(); ++m)
            if (adj[v][cand[m]]) rest.push_back(cand[m]);
        if (has_clique(adj, rest, need - 1)) return true;
    }
    return false;
}

}  // namespace

extern "C" {

// Stable ascending sort by t_ps inside each segment.  perm[k] = input index of out[k].
int oracle_sort(const Hit* in, Hit* out, uint32_t* perm, uint32_t n, const uint32_t* seg_off, uint32_t n_seg) {
    std::vector<uint32_t> idx(n);
    for (uint32_t i = 0; i < n; ++i) idx[i] = i;
    for (uint32_t s = 0; s < n_seg; ++s)
        std::stable_sort(idx.begin() + seg_off[s], idx.begin() + seg_off[s + 1],
                         [in](uint32_t a, uint32_t b) { return in[a].t_ps < in[b].t_ps; });
    for (uint32_t k = 0; k < n; ++k) {
        out[k] = in[idx[k]];
        if (perm) perm[k] = idx[k];
    }
    return 0;
}

// L1 (Q | LC), L2 (clique / star) and the ascending seed list on time-sorted hits.
// seeds must have room for n entries.  Returns 0, or -1 for invalid parameters.
int oracle_trigger(const Hit* h, uint32_t n, const uint32_t* seg_off, uint32_t n_seg, uint32_t n_pmt,
                   uint32_t n_tower, uint32_t ppt, const int32_t* pair_block, const int32_t* blocks,
                   const Params* p, uint8_t* flags, uint32_t* seeds, uint32_t* n_seeds, int32_t* status) {
    if (p->l2_multiplicity < 1 || p->lc_window_ps < 0 || p->l2_window_ps < 0) return -1;
    const Geo g{n_pmt, n_tower, ppt, pair_block, blocks};
    const uint64_t LC = (uint64_t)p->lc_window_ps, W = (uint64_t)p->l2_window_ps;
    const int N = (int)p->l2_multiplicity;
    *status = 0;
    std::memset(flags, 0, n);
    uint32_t ns = 0;
    for (uint32_t s = 0; s < n_seg; ++s) {
        const int64_t a = seg_off[s], b = seg_off[s + 1];
        // ---- L1: charge over threshold, or a same-floor hit on another PMT within LC ----
        for (int64_t i = a; i < b; ++i) {
            uint8_t f = 0;
            if (h[i].charge >= p->q_thresh) f |= F_Q;
            bool lc = false;
            for (int64_t j = i - 1; j >= a && span(h[i].t_ps, h[j].t_ps) <= LC; --j)
                if (h[j].floor == h[i].floor && h[j].pmt_id != h[i].pmt_id) lc = true;
            for (int64_t j = i + 1; j < b && span(h[j].t_ps, h[i].t_ps) <= LC; ++j)
                if (h[j].floor == h[i].floor && h[j].pmt_id != h[i].pmt_id) lc = true;
            if (lc) f |= F_LC;
            if (f) f |= F_L1;
            flags[i] = f;
        }
        // ---- L2 on the L1 hits of this segment ----
        std::vector<int64_t> l1;
        for (int64_t i = a; i < b; ++i)
            if (flags[i] & F_L1) {
                l1.push_back(i);
                if (h[i].pmt_id >= n_pmt) *status |= S_BAD_PMT;
            }
        const int64_t m = (int64_t)l1.size();
        auto edge = [&](int64_t x, int64_t y) {  // x, y index l1[]
            const Hit &hx = h[l1[x]], &hy = h[l1[y]];
            const uint64_t d = hx.t_ps > hy.t_ps ? span(hx.t_ps, hy.t_ps) : span(hy.t_ps, hx.t_ps);
            const int64_t tab = dtmax(g, hx.pmt_id, hy.pmt_id);
            if (tab < 0) return false;
            const uint64_t lim = std::min<uint64_t>((uint64_t)tab, W);
            return d <= lim;
        };
        for (int64_t x = 0; x < m; ++x) {
            std::vector<int64_t> nb;  // neighbours of x, ascending
            int64_t lo = x;
            while (lo > 0 && span(h[l1[x]].t_ps, h[l1[lo - 1]].t_ps) <= W) --lo;
            for (int64_t y = lo; y < m && (y <= x || span(h[l1[y]].t_ps, h[l1[x]].t_ps) <= W); ++y)
                if (y != x && edge(x, y)) nb.push_back(y);
            const int k = (int)nb.size();
            if (k < N - 1) continue;
            flags[l1[x]] |= F_L2STAR;
            bool l2 = true;
            if (p->l2_mode == 0) {
                std::vector<std::vector<uint8_t>> adj(k, std::vector<uint8_t>(k, 0));
                for (int u = 0; u < k; ++u)
                    for (int v = 0; v < k; ++v)
                        if (u != v) adj[u][v] = edge(nb[u], nb[v]);
                std::vector<int> cand(k);
                for (int u = 0; u < k; ++u) cand[u] = u;
                l2 = has_clique(adj, cand, N - 1);
            }
            if (l2) flags[l1[x]] |= F_L2;
        }
        // ---- seeds: ascending sorted-array indices of L2 hits ----
        for (int64_t i = a; i < b; ++i)
            if (flags[i] & F_L2) seeds[ns++] = (uint32_t)i;
    }
    *n_seeds = ns;
    return 0;
}

// Merge the [t-H, t+H] windows of consecutive seeds (closed intervals; merge iff gap <= 2H),
// never across a segment.  events must have room for n_seeds entries.
int oracle_events(const Hit* h, uint32_t n, const uint32_t* seg_off, uint32_t n_seg, const uint32_t* seeds,
                  uint32_t n_seeds, const Params* p, Event* events, uint32_t* n_events, uint8_t* flags) {
    (void)n;
    const int64_t H = p->event_half_ps;
    if (H < 0) return -1;
    uint32_t ne = 0, k = 0;
    for (uint32_t s = 0; s < n_seg; ++s) {
        const uint32_t a = seg_off[s], b = seg_off[s + 1];
        while (k < n_seeds && seeds[k] < b) {
            uint32_t first = k, last = k;
            while (last + 1 < n_seeds && seeds[last + 1] < b &&
                   span(h[seeds[last + 1]].t_ps, h[seeds[last]].t_ps) <= 2 * (uint64_t)H)
                ++last;
            // window bounds in exact arithmetic (R1: any int64 timestamp); the reported int64 fields are the exact
            // values where they fit, else modulo 2^64 (R13: unclipped)
            const __int128 ts = (__int128)h[seeds[first]].t_ps - H, te = (__int128)h[seeds[last]].t_ps + H;
            Event e;
            e.t_start = (int64_t)(uint64_t)ts;
            e.t_end = (int64_t)(uint64_t)te;
            uint32_t lo = seeds[first], hi = seeds[last] + 1;
            while (lo > a && (__int128)h[lo - 1].t_ps >= ts) --lo;  // lower_bound(t >= t_start)
            while (hi < b && (__int128)h[hi].t_ps <= te) ++hi;      // upper_bound(t <= t_end)
            e.hit_begin = lo;
            e.hit_end = hi;
            e.seed_begin = first;
            e.n_seeds = last - first + 1;
            if (flags)
                for (uint32_t i = lo; i < hi; ++i) flags[i] |= F_INEVT;
            events[ne++] = e;
            k = last + 1;
        }
    }
    *n_events = ne;
    return 0;
}

// Level-0 N-in-TW trigger on time-sorted hits (reading R14).  Inside each segment, window
// start k fires <=> hit k+N-1 exists in the segment and t[k+N-1] - t[k] < TW (strict).  l0[i] bit 0 (1) =
// i is a firing window start; bit 1 (2) = i is one of the N hits k..k+N-1 of some firing window.
// *n_start = number of firing starts.  N >= 1; TW <= 0 never fires.
int oracle_l0_ntw(const Hit* h, uint32_t n, const uint32_t* seg_off, uint32_t n_seg, uint32_t N, int64_t TW,
                  uint8_t* l0, uint32_t* n_start) {
    if (N < 1) return -1;
    for (uint32_t i = 0; i < n; ++i) l0[i] = 0;
    uint32_t count = 0;
    for (uint32_t s = 0; s < n_seg; ++s) {
        const uint64_t a = seg_off[s], b = seg_off[s + 1];
        for (uint64_t k = a; k < b; ++k) {
            const uint64_t last = k + (uint64_t)N - 1;
            if (last >= b) break;  // fewer than N hits left in the segment
            const __int128 dt = (__int128)h[last].t_ps - (__int128)h[k].t_ps;
            if (dt < (__int128)TW) {
                l0[k] |= 1;
                for (uint64_t j = k; j <= last; ++j) l0[j] |= 2;
                ++count;
            }
        }
    }
    *n_start = count;
    return 0;
}

// Pair-coincidence seeds of the paper on time-sorted hits (readings R21, R4, R5).
// For every ordered pair (i, j), j != i, of one segment with different pmt_id and |t_j - t_i| <= the rule's window
// (inclusive, R4), hit i gets
//   SC  (1): same tower (pmt_id / ppt) and adj[(pmt_i % ppt) * ppt + pmt_j % ppt] != 0   ("adjacent PMTs")
//   FC  (2): same floor field                                                       ("same floor")
//   AFC (4): same tower and floor fields that differ by exactly 1                   ("two consecutive floors")
// The scan walks outwards from i in both directions while |dt| <= the largest window.
int oracle_pair_seeds(const Hit* h, uint32_t n, const uint32_t* seg_off, uint32_t n_seg, uint32_t ppt,
                      const uint8_t* adj, int64_t w_sc, int64_t w_fc, int64_t w_afc, uint8_t* bits) {
    if (ppt < 1 || w_sc < 0 || w_fc < 0 || w_afc < 0) return -1;
    for (uint32_t i = 0; i < n; ++i) bits[i] = 0;
    const int64_t wmax = std::max(w_sc, std::max(w_fc, w_afc));
    auto rules = [&](const Hit& a, const Hit& b, __int128 dt) -> uint8_t {
        if (a.pmt_id == b.pmt_id) return 0;
        uint8_t m = 0;
        const bool same_tower = a.pmt_id / ppt == b.pmt_id / ppt;
        if (dt <= w_sc && same_tower && adj[(size_t)(a.pmt_id % ppt) * ppt + b.pmt_id % ppt]) m |= 1;
        if (dt <= w_fc && a.floor == b.floor) m |= 2;
        const int df = (int)a.floor - (int)b.floor;
        if (dt <= w_afc && same_tower && (df == 1 || df == -1)) m |= 4;
        return m;
    };
    for (uint32_t s = 0; s < n_seg; ++s) {
        const int64_t a = seg_off[s], b = seg_off[s + 1];
        for (int64_t i = a; i < b; ++i) {
            uint8_t m = 0;
            for (int64_t j = i - 1; j >= a; --j) {
                const __int128 dt = (__int128)h[i].t_ps - (__int128)h[j].t_ps;
                if (dt > wmax) break;
                m |= rules(h[i], h[j], dt);
            }
            for (int64_t j = i + 1; j < b; ++j) {
                const __int128 dt = (__int128)h[j].t_ps - (__int128)h[i].t_ps;
                if (dt > wmax) break;
                m |= rules(h[i], h[j], dt);
            }
            bits[i] = m;
        }
    }
    return 0;
}

// The paper's combined trigger (reading R22): for every firing level-0 window start k (l0[k] & 1; its
// N hits k..k+N-1 lie in one segment), OR the pair bits of the N hits; out[k] gets 8 when both SC and AFC occur among
// them ("N7TW with [SC and AFC]") and 16 when both FC and AFC occur ("N7TW with [FC and AFC]").  Other hits get 0.
int oracle_l0_combine(const uint8_t* l0, const uint8_t* pair_bits, uint32_t n, uint32_t N, uint8_t* out) {
    if (N < 1) return -1;
    for (uint32_t k = 0; k < n; ++k) {
        out[k] = 0;
        if (!(l0[k] & 1)) continue;
        if ((uint64_t)k + N > n) return -2;  // a start bit without its window: not an output of oracle_l0_ntw
        uint8_t m = 0;
        for (uint32_t j = k; j < k + N; ++j) m |= pair_bits[j];
        if ((m & 1) && (m & 4)) out[k] |= 8;
        if ((m & 2) && (m & 4)) out[k] |= 16;
    }
    return 0;
}

// Distinct-PMT level-0 trigger (reading R23).  Inside each segment, window start k fires <=> the hits
// j >= k with t_j - t_k < TW (strict, as for N-in-TW) carry at least N different pmt_id values.  Its members are the
// hits k..e_k, e_k = the first hit at which the N-th different PMT appears (with all PMTs different this is the plain
// N-in-TW window k..k+N-1).  l0[i]: 1 = firing start, 2 = member of some firing window; *n_start = firing starts.
int oracle_l0_dntw(const Hit* h, uint32_t n, const uint32_t* seg_off, uint32_t n_seg, uint32_t N, int64_t TW,
                   uint8_t* l0, uint32_t* n_start) {
    if (N < 1) return -1;
    for (uint32_t i = 0; i < n; ++i) l0[i] = 0;
    uint32_t count = 0;
    std::vector<uint16_t> seen;
    for (uint32_t s = 0; s < n_seg; ++s) {
        const uint64_t a = seg_off[s], b = seg_off[s + 1];
        for (uint64_t k = a; k < b; ++k) {
            seen.clear();
            for (uint64_t j = k; j < b; ++j) {
                const __int128 dt = (__int128)h[j].t_ps - (__int128)h[k].t_ps;
                if (!(dt < (__int128)TW)) break;
                if (std::find(seen.begin(), seen.end(), h[j].pmt_id) == seen.end()) seen.push_back(h[j].pmt_id);
                if (seen.size() == N) {
                    l0[k] |= 1;
                    for (uint64_t m = k; m <= j; ++m) l0[m] |= 2;
                    ++count;
                    break;
                }
            }
        }
    }
    *n_start = count;
    return 0;
}

// ---- NEXT-3: the paper's CPU preparation.  Raw hit k = a 16-byte header {t_ps, pmt_id, floor,
// n_samples, pad} and n_samples 16-bit waveform samples; the waveforms of all hits are concatenated in hit order, so
// hit k's samples start at the sum of the sample counts before it.  charge = sum of the samples, saturated at 65535;
// samples that would lie behind the waveform section count as 0 and set status bit 32.  Output: fixed-size records,
// slice-major then PMT-major, arrival order kept inside a (slice, PMT) run; run_off[slice * n_pmt + pmt] .. =
// offsets of the runs.  A hit with pmt_id >= n_pmt sets status bit 8 and is filed under the last PMT of its slice.
struct RawHit {
    int64_t t_ps;
    uint16_t pmt_id, floor, n_samples, pad;
};
static_assert(sizeof(RawHit) == 16, "raw header is 16 bytes");

int oracle_prepare(const RawHit* raw, const uint16_t* samples, uint32_t n_raw, uint32_t n_samples_total,
                   const uint32_t* slice_off, uint32_t n_slices, uint32_t n_pmt, Hit* out, uint32_t* run_off,
                   int32_t* status) {
    if (n_pmt < 1 || n_slices < 1) return -1;
    *status = 0;
    // waveform start of every hit
    std::vector<uint64_t> woff(n_raw + 1, 0);
    for (uint32_t k = 0; k < n_raw; ++k) woff[k + 1] = woff[k] + raw[k].n_samples;
    uint32_t pos = 0;
    for (uint32_t s = 0; s < n_slices; ++s)
        for (uint32_t p = 0; p < n_pmt; ++p) {
            run_off[(uint64_t)s * n_pmt + p] = pos;
            for (uint32_t k = slice_off[s]; k < slice_off[s + 1]; ++k) {
                uint32_t q = raw[k].pmt_id;
                if (q >= n_pmt) { *status |= 8; q = n_pmt - 1; }
                if (q != p) continue;
                uint64_t sum = 0;
                for (uint32_t j = 0; j < raw[k].n_samples; ++j) {
                    const uint64_t at = woff[k] + j;
                    if (at >= n_samples_total) { *status |= 32; continue; }
                    sum += samples[at];
                }
                Hit h;
                h.t_ps = raw[k].t_ps;
                h.pmt_id = raw[k].pmt_id;
                h.floor = raw[k].floor;
                h.charge = (uint16_t)(sum > 65535 ? 65535 : sum);
                h.pad = raw[k].pad;
                out[pos++] = h;
            }
        }
    run_off[(uint64_t)n_slices * n_pmt] = pos;
    return 0;
}

}  // extern "C"
