// pat_api.cu -- the C-ABI of include/pat.h: argument checking, workspace layout, plan state,
// stream-ordered orchestration of the kernels.  No arithmetic of the method runs on the host.
#include "pat_internal.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <numeric>

namespace {

thread_local std::string g_create_error;   // last pat_plan_create failure of THIS thread (plan == NULL in pat_last_error)

// ---- cross-call overlap: the launch chain ------------------------------------------------------------------
// One frame of configs[1] is ~10 us of GPU work: between two calls the launch gap, the gather's prologue and the
// ragged end of its CTAs are a third of that.  Inside a stream capture (CUDA graph) consecutive calls are therefore
// NOT captured as one linear chain.  With P_j / G_j the pre-pass / gather node of call j of an uninterrupted run
// of calls on the capturing stream, the edges are
//     G_{j-1} --programmatic--> G_j    the CTAs of G_j take the SM slots the CTAs of G_{j-1} free one by one, and
//                                      stream the table beside the draining G_{j-1};
//     P_j     --full----------> G_j    b (and the zeroed images) are complete before G_j starts;
//     G_{j-3}, P_{j-1} --full-> P_j    and NO edge from G_{j-1}, G_{j-2}: the pre-pass of call j runs while the two
//                                      gathers before it are still busy, so its latency (a trip to HBM behind the table
//                                      stream, ~4 us) is off the critical path.  (The edge from P_{j-1} keeps the
//                                      pre-passes one ordered chain, which is how the graph executor runs them early.)
// What makes that safe is carried by those edges alone:
//   * b is triple-buffered per plan (calls rotate through three buffers): P_j writes the buffer G_{j-3} read, and
//     G_{j-3} has completed; G_{j-1} and G_{j-2} read the other two;
//   * G_j needs P_j, hence G_{j-3}: at most three gathers of a run are ever in flight, and they only READ shared
//     data (table, work list) and accumulate into their own images;
//   * the host allows the edges only if nothing foreign sits between the calls -- the capture's dependency set at
//     call j is exactly {G_{j-1}} -- and if the images and traces of call j do not overlap the images of call j-1
//     (P_j zeroes them while that gather may still accumulate); if they overlap those of call j-2 (a caller
//     alternating between two image buffers), P_j hangs on G_{j-2} instead of G_{j-3}.  Everything enqueued before
//     the run is ordered before P_0, hence before every node of the run; whatever is captured after call j depends
//     on G_j, and one thread of every gather executes griddepcontrol.wait before the grid finishes, so the
//     completion of G_j implies the completion of G_{j-1} (and so on down the run).
// Any other call -- outside a capture, host buffers, overlapping images, foreign work in between -- is captured /
// launched the ordinary way (P then G in stream order, G's prologue overlapping P through a programmatic launch).
struct ChainCall {
    cudaGraphNode_t gather;
    uintptr_t img_lo, img_hi;
};
struct ChainRun {
    unsigned long long capture_id = 0;
    cudaGraphNode_t head_prepass = nullptr;     // P_{j-1}: the latest pre-pass of the run (P_j hangs on it as well,
                                                // which keeps the pre-passes one ordered chain beside the gathers)
    std::vector<ChainCall> calls;               // the last (up to) three calls of the run, oldest first
};
std::mutex g_chain_mu;
std::vector<ChainRun> g_chain;            // one entry per capture in progress (bounded, oldest dropped)

bool capture_deps(cudaStream_t st, unsigned long long *id, cudaGraphNode_t *node) {
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    const cudaGraphNode_t *deps = nullptr;
    const cudaGraphEdgeData *edges = nullptr;
    size_t nd = 0;
    if (cudaStreamGetCaptureInfo_v3(st, &cs, id, nullptr, &deps, &edges, &nd) != cudaSuccess) { cudaGetLastError(); return false; }
    if (cs != cudaStreamCaptureStatusActive) { *id = 0; return false; }
    if (nd != 1 || !deps) return false;
    *node = deps[0];
    return true;
}

ChainRun *find_run(unsigned long long id) {
    for (ChainRun &r : g_chain)
        if (r.capture_id == id) return &r;
    return nullptr;
}

// Decision for the call about to be captured.  chained: the node P_j must depend on (pre_dep) and G_{j-1}.
struct ChainPlan {
    bool chained = false;
    unsigned long long capture_id = 0;
    cudaGraphNode_t pre_dep = nullptr, prev_gather = nullptr, bound_dep = nullptr;   // bound_dep: G_{j-3} or NULL
};
ChainPlan chain_begin(cudaStream_t st, const void *traces, size_t tbytes, const void *images, size_t ibytes, int depth) {
    ChainPlan cp;
    cudaGraphNode_t node = nullptr;
    const bool single = capture_deps(st, &cp.capture_id, &node);
    if (!cp.capture_id) return cp;                                // not capturing
    std::lock_guard<std::mutex> lk(g_chain_mu);
    ChainRun *r = find_run(cp.capture_id);
    if (!single || !r || r->calls.empty() || r->calls.back().gather != node) return cp;
    const uintptr_t i0 = (uintptr_t)images, i1 = i0 + ibytes, t0 = (uintptr_t)traces, t1 = t0 + tbytes;
    const size_t n = r->calls.size();
    auto clash = [&](const ChainCall &c) {
        return !(i1 <= c.img_lo || c.img_hi <= i0) || !(t1 <= c.img_lo || c.img_hi <= t0);
    };
    if (clash(r->calls[n - 1])) return cp;                        // G_{j-1} will still be running: ordinary capture
    cp.chained = true;
    cp.prev_gather = node;
    // images alternating between two buffers (A, B, A, ...): P_j zeroes what G_{j-2} wrote, so it waits for that one
    if (n >= 2 && (depth <= 2 || clash(r->calls[n - 2]))) cp.bound_dep = r->calls[n - 2].gather;
    else cp.bound_dep = n >= 3 ? r->calls[n - 3].gather : nullptr;
    cp.pre_dep = r->head_prepass;
    return cp;
}

// After the launches of a call inside a capture: extend the run, or start a new one at this call.
void chain_commit(const ChainPlan &cp, cudaGraphNode_t prepass, cudaGraphNode_t gather, const void *images, size_t ibytes) {
    if (!cp.capture_id) return;
    std::lock_guard<std::mutex> lk(g_chain_mu);
    ChainRun *r = find_run(cp.capture_id);
    if (!r) {
        if (g_chain.size() >= 16) g_chain.erase(g_chain.begin());
        g_chain.emplace_back();
        r = &g_chain.back();
        r->capture_id = cp.capture_id;
    }
    if (!cp.chained) r->calls.clear();
    r->head_prepass = prepass;
    if (!gather || !r->head_prepass) { r->calls.clear(); r->head_prepass = nullptr; return; }   // nothing to chain behind
    r->calls.push_back(ChainCall{gather, (uintptr_t)images, (uintptr_t)images + ibytes});
    if (r->calls.size() > 3) r->calls.erase(r->calls.begin());
}

cudaError_t set_capture_deps(cudaStream_t st, cudaGraphNode_t full_a, cudaGraphNode_t full_b, cudaGraphNode_t programmatic) {
    cudaGraphNode_t nodes[3];
    cudaGraphEdgeData edges[3];
    std::memset(edges, 0, sizeof(edges));
    size_t n = 0;
    if (full_a) nodes[n++] = full_a;
    if (full_b && full_b != full_a) nodes[n++] = full_b;
    if (programmatic) {
        edges[n].from_port = cudaGraphKernelNodePortProgrammatic;
        edges[n].type = cudaGraphDependencyTypeProgrammatic;
        nodes[n++] = programmatic;
    }
    return cudaStreamUpdateCaptureDependencies_v2(st, nodes, edges, n, cudaStreamSetCaptureDependencies);
}

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

pat_status fail(pat_plan *p, pat_status st, const std::string &msg) {
    if (p) p->err = msg; else g_create_error = msg;
    return st;
}
pat_status cuda_fail(pat_plan *p, int e, const char *what) {
    std::string m = std::string(what) + ": " + cudaGetErrorString((cudaError_t)e);
    cudaGetLastError();                // clear the sticky-less error state
    return fail(p, PAT_ERR_CUDA, m);
}

bool dims_ok(const pat_grid *g, int32_t nsens, int64_t npix, int32_t nt, int32_t max_batch) {
    if (!g || (g->ndim != 2 && g->ndim != 3)) return false;
    int64_t N = 1;
    for (int d = 0; d < g->ndim; ++d) {
        if (g->n[d] < 2) return false;
        N *= g->n[d];
        if (N > (int64_t)INT32_MAX) return false;
    }
    if (!(g->h > 0.0f) || !std::isfinite(g->h)) return false;
    if (nsens <= 0 || npix <= 0 || npix > N || nt < 2 || max_batch < 1) return false;
    if ((int64_t)nt > (1 << 22)) return false;              // k is recovered from a 2^23-biased float
    return true;
}

// Is `p` device memory?  1 = device/managed, 0 = host (pinned or pageable), -1 = query failed.
int is_device_ptr(const void *p) {
    cudaPointerAttributes a{};
    cudaError_t e = cudaPointerGetAttributes(&a, p);
    if (e != cudaSuccess) { cudaGetLastError(); return -1; }
    return (a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged) ? 1 : 0;
}

// 64-bit Morton key of a node (x fastest); keeps 256 consecutive ROI pixels spatially compact.
inline uint64_t spread2(uint32_t v) {
    uint64_t x = v;
    x = (x | (x << 16)) & 0x0000FFFF0000FFFFull;
    x = (x | (x << 8)) & 0x00FF00FF00FF00FFull;
    x = (x | (x << 4)) & 0x0F0F0F0F0F0F0F0Full;
    x = (x | (x << 2)) & 0x3333333333333333ull;
    x = (x | (x << 1)) & 0x5555555555555555ull;
    return x;
}
inline uint64_t spread3(uint32_t v) {
    uint64_t x = v & 0x1FFFFF;
    x = (x | (x << 32)) & 0x1F00000000FFFFull;
    x = (x | (x << 16)) & 0x1F0000FF0000FFull;
    x = (x | (x << 8)) & 0x100F00F00F00F00Full;
    x = (x | (x << 4)) & 0x10C30C30C30C30C3ull;
    x = (x | (x << 2)) & 0x1249249249249249ull;
    return x;
}

// Samples [lo, hi) of a trace that the rows of `meta` ({kmin, kmax | flags} per row) can touch: b[kmin .. kmax+1],
// i.e. p[kmin-1 .. kmax+2] with the central difference, rounded outwards to whole 16-byte quads.
void needed_samples(const std::vector<int32_t> &meta, int32_t nt, int32_t *lo, int32_t *hi) {
    int32_t kmin = INT32_MAX, kmax = -1;
    for (size_t r = 0; r + 1 < meta.size(); r += 2) {
        const int32_t a = meta[r], b = meta[r + 1] < 0 ? -1 : (meta[r + 1] & 0x3FFFFFFF);
        if (b < a) continue;
        kmin = std::min(kmin, a);
        kmax = std::max(kmax, b);
    }
    if (kmax < 0) { *lo = *hi = 0; return; }                // no valid entry at all: nothing is read
    *lo = std::max(0, kmin - 1) & ~3;
    *hi = std::min(nt, (kmax + 3 + 3) & ~3);
}

// Device memory of the plan beyond its workspace: from the caller's provider (alloc.cu), accounted per plan.
bool plan_alloc(pat_plan *p, size_t bytes, PatDevBuf *out) {
    return pat_dev_alloc(p->alloc, bytes, out, &p->dev_bytes, &p->dev_bytes_peak);
}
void plan_free(pat_plan *p, PatDevBuf *buf) { pat_dev_free(p->alloc, buf, &p->dev_bytes); }

void drop_schedules(pat_plan *p) {
    for (PatSchedule &sc : p->schedules) plan_free(p, &sc.buf);
    p->schedules.clear();
}

// The table is complete: reduce every (tile, sensor) row to its k-range and keep a host copy,
// from which the per-configuration work lists are built (build_schedule).  Synchronises `stream`.
pat_status finalize_table(pat_plan *p, void *stream) {
    const int64_t nrows = p->dims.ntiles * p->dims.nsens;
    PatLaunchCtx ctx{stream, p->num_sms, false};
    int e = pat_launch_row_meta(ctx, (const float *)(p->ws + p->lay.tau), p->ws + p->lay.meta, nrows, p->dims.nt);
    if (e) return cuda_fail(p, e, "row-meta launch");
    ++p->launches;
    try { p->host_meta.resize((size_t)nrows * 2); } catch (...) { return fail(p, PAT_ERR_NOMEM, "host allocation failed"); }
    cudaError_t ce = cudaMemcpyAsync(p->host_meta.data(), p->ws + p->lay.meta, (size_t)nrows * 2 * sizeof(int32_t),
                                     cudaMemcpyDeviceToHost, (cudaStream_t)stream);
    if (ce == cudaSuccess) ce = cudaStreamSynchronize((cudaStream_t)stream);
    if (ce != cudaSuccess) return cuda_fail(p, ce, "row-meta read-back");
    p->meta_valid = true;
    needed_samples(p->host_meta, p->dims.nt, &p->need_lo, &p->need_hi);
    return PAT_OK;
}

struct Entry { int32_t x, y, z, w; };       // one int4 of the work list (layout: gather.cu)
struct Slot { int32_t row, sensor, s0, klen, len; bool whole, allvalid; };

// Work list for one shared-memory geometry.  Every row with a valid pixel is cut into segments of
// at most wr-4 k-values (one slot each; rows without a valid pixel vanish).  Slots are dealt to
// grid_x persistent CTAs in equal shares and grouped into chunks of at most R slots that share a
// tile and whose sample windows all lie inside one frame [cbase, cbase + wr) -- the window of a slot
// is then ONE bulk copy to offset (s0 - cbase) and the consumers index it with k - cbase.
// Chunk flags: simple = R whole rows (no per-slot range check needed); contig = the slots' u rows
// are consecutive in the table (one bulk copy for the whole chunk).
pat_status build_schedule(pat_plan *p, const PatGatherConfig &cfg, PatSchedule **out) {
    const int64_t ntiles = p->dims.ntiles;
    const int32_t S = p->dims.nsens;
    const int32_t step = cfg.step, R = cfg.R;
    const bool blocked = pat_gather_blocked(cfg.bp);   // window units: 32-sample blocks (else samples)
    const int32_t amask = blocked ? ~31 : ~3, ntb = (p->dims.nt + 31) / 32;
    const int32_t *meta = cfg.onfly ? p->onfly_meta.data() : p->host_meta.data();
    if ((int64_t)S * p->nt4 > (int64_t)INT32_MAX) return fail(p, PAT_ERR_UNSUPPORTED, "nsens*nt exceeds 2^31");
    int64_t V = 0;
    for (int64_t r = 0; r < ntiles * S; ++r) {
        if (!p->tile_active.empty() && !p->tile_active[(size_t)(r / S)]) continue;
        const int32_t kmin = meta[2 * r], kmax = meta[2 * r + 1] < 0 ? -1 : (meta[2 * r + 1] & 0x3FFFFFFF);
        if (kmax >= kmin) V += (kmax + 1 - (kmin & amask) + step - 1) / step;
    }
    PatSchedule sc;
    sc.cfg = cfg;
    int per_sm = 0;
    int e = pat_gather_occupancy(cfg, &per_sm);
    if (e) return cuda_fail(p, e, "gather occupancy query");
    if (per_sm < 1) return fail(p, PAT_ERR_CUDA, "gather kernel does not fit on an SM with this tuning");
    int64_t G = (int64_t)p->num_sms * per_sm;
    sc.grid_x = 0;
    if (V == 0) { p->schedules.push_back(sc); *out = &p->schedules.back(); return PAT_OK; }
    std::vector<Entry> list;
    std::vector<int32_t> cta_chunk;
    std::vector<int32_t> cost;                       // per chunk: fixed part + slots
    const int32_t chunk_cost = p->env.chunk_cost;
    const int32_t slow_cost = p->env.slow_cost;      // a slot of a checked chunk, in units of half a fast slot
    const size_t per_chunk = (size_t)R + 1;
    try {
        list.reserve((size_t)(V / R + ntiles + 16) * per_chunk);
        std::vector<Slot> cur, rest;
        int32_t cur_tile = -1, used = 0;             // used = window samples already packed into the chunk
        auto close_chunk = [&]() {
            if (cur.empty()) return;
            bool fast = true, contig = true;
            for (size_t q = 0; q < cur.size(); ++q) {
                fast = fast && cur[q].whole && cur[q].allvalid;
                contig = contig && cur[q].row == cur[0].row + (int32_t)q;
            }
            if (cfg.onfly) contig = true;              // no u copies at all: the consumers compute u
            const int32_t flags = (fast ? 1 : 0) | (contig ? 2 : 0) | ((int32_t)cur.size() << 8);
            list.push_back(Entry{cur_tile, 0, flags, cur[0].row});
            int32_t pos = 0;
            for (const Slot &sl : cur) {
                list.push_back(Entry{sl.row, blocked ? sl.sensor * ntb + (sl.s0 >> 5) : sl.sensor * p->nt4 + sl.s0,
                                     (int32_t)((uint32_t)pos | ((uint32_t)sl.klen << 16) | (contig ? 0x80000000u : 0u)),
                                     sl.s0});
                pos += sl.len;
            }
            for (int32_t q = (int32_t)cur.size(); q < R; ++q) list.push_back(Entry{0, 0, 0, 0});
            // cost model (measured with the per-CTA timeline, PAT_TRACE_FILE): bytes moved -- 256 samples
            // of u per slot plus its window -- plus a fixed part per chunk; checked chunks cost more per slot
            // Bp <= 2 (HBM-bound).  For larger Bp the time goes with rows x frames (shared-memory bound).
            int32_t cc = chunk_cost * 64;
            if (cfg.bp <= 2)
                for (const Slot &sl : cur) cc += (256 + sl.len) * (fast ? 2 : slow_cost) / 2;
            else
                cc += 128 * (int32_t)cur.size() * (fast ? 2 : 3);
            cost.push_back(cc);
            cur.clear();
            used = 0;
        };
        auto add_slot = [&](int32_t t, const Slot &sl) {
            if (!cur.empty() && (cur_tile != t || (int32_t)cur.size() == R || used + sl.len > cfg.cap)) close_chunk();
            cur_tile = t;
            used += sl.len;
            cur.push_back(sl);
        };
        for (int64_t t = 0; t < ntiles; ++t) {
            if (!p->tile_active.empty() && !p->tile_active[(size_t)t]) continue;   // pat_set_roi_mask
            rest.clear();
            // whole rows in sensor order (their u rows stay consecutive: one bulk copy per chunk) ...
            for (int32_t s = 0; s < S; ++s) {
                const int64_t r = t * S + s;
                const int32_t kmin = meta[2 * r], kmax = meta[2 * r + 1] < 0 ? -1 : (meta[2 * r + 1] & 0x3FFFFFFF);
                if (kmax < kmin) continue;
                const bool allvalid = (meta[2 * r + 1] >> 30) & 1;
                const int32_t n0 = kmin & amask, kend = kmax + 1;
                // window of a slot with k-range [s0, s0+klen): samples s0 .. s0+klen, in units
                auto units = [&](int32_t s0, int32_t klen) {
                    return blocked ? ((s0 + klen) >> 5) - (s0 >> 5) + 1 : (klen + 4) & ~3;
                };
                if (kend - n0 <= step) {
                    add_slot((int32_t)t, Slot{(int32_t)r, s, n0, kend - n0, units(n0, kend - n0), true, allvalid});
                } else {
                    for (int32_t s0 = n0; s0 < kend; s0 += step) {
                        const int32_t klen = std::min(step, kend - s0);
                        rest.push_back(Slot{(int32_t)r, s, s0, klen, units(s0, klen), false, false});
                    }
                }
            }
            // ... then the segments of the long rows
            for (const Slot &sl : rest) add_slot((int32_t)t, sl);
            close_chunk();
        }
        // deal whole chunks to the CTAs in contiguous, equal-cost shares
        const int64_t nchunks = (int64_t)cost.size();
        G = std::min<int64_t>(G, nchunks);
        sc.grid_x = (int)G;
        int64_t total = 0;
        for (int32_t cc : cost) total += cc;
        cta_chunk.reserve((size_t)G + 1);
        cta_chunk.push_back(0);
        int64_t q = 0, acc = 0;                     // acc = cost of chunks [0, q)
        for (int64_t c = 1; c < G; ++c) {
            const int64_t want = total * c / G;
            const int64_t qmin = cta_chunk.back() + 1, qmax = nchunks - (G - c);
            while (q < qmax && (q < qmin || acc + cost[q] / 2 < want)) acc += cost[q++];
            cta_chunk.push_back((int32_t)q);
        }
        cta_chunk.push_back((int32_t)nchunks);
    } catch (...) { return fail(p, PAT_ERR_NOMEM, "host allocation failed"); }
    if (list.size() / per_chunk > (size_t)INT32_MAX) return fail(p, PAT_ERR_UNSUPPORTED, "work list too long");
    sc.nchunks = (int64_t)(list.size() / per_chunk);
    if (!p->env.sched_dump.empty()) {                            // diagnostic: per-CTA share composition
        if (FILE *f = std::fopen(p->env.sched_dump.c_str(), "w")) {
            for (int64_t c = 0; c < G; ++c) {
                int64_t nch = cta_chunk[c + 1] - cta_chunk[c], nsl = 0, nwin = 0, nfast = 0;
                for (int64_t q = cta_chunk[c]; q < cta_chunk[c + 1]; ++q) {
                    const Entry *h = &list[(size_t)q * per_chunk];
                    nfast += h->z & 1;
                    for (int v = 1; v <= R; ++v) {
                        const uint32_t klen = ((uint32_t)h[v].z >> 16) & 0x7FFFu;
                        if (klen) { ++nsl; nwin += (klen + 4) & ~3; }
                    }
                }
                std::fprintf(f, "%lld %lld %lld %lld %lld\n", (long long)c, (long long)nch, (long long)nsl, (long long)nwin, (long long)nfast);
            }
            std::fclose(f);
        }
    }
    {
        if (p->env.debug) {
            int64_t ns = 0, nc = 0, nreal = 0;
            for (size_t q = 0; q < list.size(); q += per_chunk) {
                ns += list[q].z & 1; nc += (list[q].z >> 1) & 1; nreal += list[q].z >> 8;
            }
            std::fprintf(stderr, "[pat] schedule bp=%d wr=%d R=%d stages=%d: grid=%d slots=%lld chunks=%lld "
                         "(fast %lld, contig %lld, slots/chunk %.2f) smem=%zu B, %d CTA/SM\n", cfg.bp, cfg.wr, R,
                         cfg.stages, sc.grid_x, (long long)V, (long long)sc.nchunks, (long long)ns, (long long)nc,
                         (double)nreal / (double)sc.nchunks, pat_gather_smem_bytes(cfg), per_sm);
        }
    }
    const size_t main_entries = list.size();
    try {                                                        // every CTA's first chunk once more, indexed by CTA
        for (int64_t c = 0; c < G; ++c)
            for (size_t q = 0; q < per_chunk; ++q) list.push_back(list[(size_t)cta_chunk[(size_t)c] * per_chunk + q]);
    } catch (...) { return fail(p, PAT_ERR_NOMEM, "host allocation failed"); }
    // one block from the caller's provider: [chunk entries][first-chunk copies][CTA ranges]
    const size_t list_bytes = list.size() * sizeof(Entry);
    if (!plan_alloc(p, list_bytes + cta_chunk.size() * sizeof(int32_t), &sc.buf))
        return fail(p, PAT_ERR_NOMEM, "work list: the device-memory provider returned nothing");
    sc.d_sched = sc.buf.p;
    sc.d_first = (char *)sc.buf.p + main_entries * sizeof(Entry);
    sc.d_cta_chunk = (int32_t *)((char *)sc.buf.p + list_bytes);
    cudaError_t ce = cudaMemcpy(sc.d_sched, list.data(), list_bytes, cudaMemcpyHostToDevice);
    if (ce == cudaSuccess)
        ce = cudaMemcpy(sc.d_cta_chunk, cta_chunk.data(), cta_chunk.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (ce != cudaSuccess) {
        plan_free(p, &sc.buf);
        return cuda_fail(p, ce, "work-list upload");
    }
    p->schedules.push_back(sc);
    *out = &p->schedules.back();
    return PAT_OK;
}

// Every device-side call of a plan must run with the plan's device current: its workspace, work lists and streams
// belong to it, and memory from the provider would otherwise come from another device.
pat_status check_device(pat_plan *p) {
    int cur = -1;
    cudaError_t e = cudaGetDevice(&cur);
    if (e != cudaSuccess) return cuda_fail(p, e, "cudaGetDevice");
    if (cur != p->device)
        return fail(p, PAT_ERR_INVALID_ARG, "the current CUDA device is not the one the plan was created on (cudaSetDevice first)");
    return PAT_OK;
}

pat_status get_schedule(pat_plan *p, int bp, bool onfly, PatSchedule **out) {
    for (PatSchedule &sc : p->schedules)
        if (sc.cfg.bp == bp && sc.cfg.onfly == onfly) { *out = &sc; return PAT_OK; }
    const auto t_begin = std::chrono::steady_clock::now();
    struct Timer {
        pat_plan *p; std::chrono::steady_clock::time_point t0;
        ~Timer() { p->sched_build_seconds += std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count(); ++p->sched_builds; }
    } timer{p, t_begin};
    PatGatherConfig cfg = pat_gather_config(bp, p->tune_wr, p->tune_R, p->tune_stages, onfly, p->exact,
                                            p->d_w_t != nullptr, p->env);
    // the occupancy the work list is cut for is that of the kernel that will run (ensure_onfly came first)
    cfg.fastu = onfly && bp == 1 && !p->exact && !p->d_w_t && p->grid.ndim == 2 && p->t0 == 0.0f &&
                p->onfly_d2_in_range && !p->env.no_fast_delays;
    return build_schedule(p, cfg, out);
}

// Conventional BP set-up: node coordinates of every tile slot and the sensors on the device (once), and the
// k-range of every (tile, sensor) row for this c0 (a kernel with the gather's own arithmetic; synchronises).
pat_status ensure_onfly(pat_plan *p, float c0, float c0_hi, void *stream, PatOnfly *out) {   // c0 <= c0_hi: a sweep's range
    const int64_t slots = p->dims.ntiles * kTilePix;
    const int32_t S = p->dims.nsens;
    cudaStream_t st = (cudaStream_t)stream;
    if (!p->d_pix) {
        std::vector<float> pix;
        try { pix.assign((size_t)slots * 3, 0.0f); } catch (...) { return fail(p, PAT_ERR_NOMEM, "host allocation failed"); }
        const int64_t n0 = p->grid.n[0], n1 = p->grid.n[1];
        const float h = p->grid.h;
        for (int64_t sl = 0; sl < slots; ++sl) {
            int32_t pos = p->host_perm[(size_t)sl];
            if (pos < 0) pos = p->host_perm[(size_t)(sl / kTilePix * kTilePix)];      // padding: the tile's first pixel
            const int64_t q = p->roi.empty() ? pos : p->roi[(size_t)pos];
            const int64_t id[3] = {q % n0, (q / n0) % n1, q / (n0 * n1)};
            for (int dd = 0; dd < 3; ++dd) {
                volatile float stepv = (float)id[dd] * h;                            // two roundings, no contraction
                pix[(size_t)dd * slots + sl] = dd < p->grid.ndim ? p->grid.origin[dd] + stepv : 0.0f;
            }
        }
        const size_t pix_bytes = align_up(pix.size() * sizeof(float), 256);
        if (!plan_alloc(p, pix_bytes + (size_t)S * 3 * sizeof(float), &p->onfly_buf))
            return fail(p, PAT_ERR_NOMEM, "conventional BP geometry: the device-memory provider returned nothing");
        p->d_pix = (float *)p->onfly_buf.p;
        p->d_sens = (float *)((char *)p->onfly_buf.p + pix_bytes);
        cudaError_t e = cudaMemcpy(p->d_pix, pix.data(), pix.size() * sizeof(float), cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemcpy(p->d_sens, p->sensors.data(), (size_t)S * 3 * sizeof(float), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) {
            plan_free(p, &p->onfly_buf);
            p->d_pix = p->d_sens = nullptr;
            return cuda_fail(p, e, "conventional BP geometry upload");
        }
    }
    out->pix = p->d_pix; out->sens = p->d_sens; out->pix_stride = slots;
    out->inv_c0 = 1.0f / c0; out->t0 = p->t0; out->fs = p->fs; out->ndim = p->grid.ndim;
    if (p->onfly_c0 != c0 || p->onfly_c0_hi != c0_hi || p->onfly_meta.empty()) {
        const int64_t nrows = p->dims.ntiles * S;
        // scratch for the row ranges: the workspace's meta array is the table path's; same size, own block
        PatDevBuf mbuf;
        if (!plan_alloc(p, (size_t)nrows * 8 + 256, &mbuf))
            return fail(p, PAT_ERR_NOMEM, "conventional BP row ranges: the device-memory provider returned nothing");
        void *d_meta = mbuf.p;
        int32_t *d_bad = (int32_t *)((char *)mbuf.p + (size_t)nrows * 8);        // any |r - s|^2 outside the fast range?
        cudaError_t e = cudaMemsetAsync(d_bad, 0, sizeof(int32_t), st);
        PatLaunchCtx ctx{stream, p->num_sms, false};
        int le = e == cudaSuccess ? pat_launch_onfly_meta(ctx, *out, S, d_meta, nrows, p->dims.nt, d_bad) : (int)e;
        int32_t bad = 1;
        if (!le) e = cudaMemcpyAsync(&bad, d_bad, sizeof(int32_t), cudaMemcpyDeviceToHost, st);
        ++p->launches;
        try { p->onfly_meta.resize((size_t)nrows * 2); } catch (...) { cudaStreamSynchronize(st); plan_free(p, &mbuf); return fail(p, PAT_ERR_NOMEM, "host allocation failed"); }
        if (!le) e = cudaMemcpyAsync(p->onfly_meta.data(), d_meta, (size_t)nrows * 8, cudaMemcpyDeviceToHost, st);
        if (!le && e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (!le && e == cudaSuccess && c0_hi != c0) {
            // a sweep over [c0, c0_hi]: the delay of a (pixel, sensor) pair falls monotonically with the speed, so the
            // samples it can touch over the whole range lie between its k at c0_hi and its k at c0 -- the envelope
            // of the two row ranges; a row is all-valid over the range if it is at both ends
            std::vector<int32_t> hi_meta;
            try { hi_meta.resize((size_t)nrows * 2); } catch (...) { le = (int)cudaErrorMemoryAllocation; }
            PatOnfly o2 = *out;
            o2.inv_c0 = 1.0f / c0_hi;
            if (!le) le = pat_launch_onfly_meta(ctx, o2, S, d_meta, nrows, p->dims.nt);
            ++p->launches;
            if (!le) e = cudaMemcpyAsync(hi_meta.data(), d_meta, (size_t)nrows * 8, cudaMemcpyDeviceToHost, st);
            if (!le && e == cudaSuccess) e = cudaStreamSynchronize(st);
            if (!le && e == cudaSuccess) {
                // onfly_meta holds the ranges at the LOWEST speed (longest delays), hi_meta at the highest.  A pixel
                // beyond the record at the lowest speed comes into it somewhere in between with k up to nt-2, and
                // (only if t0 > 0) a pixel before the record at the highest speed enters it with k from 0.
                const int32_t kend = p->dims.nt - 2;
                const bool early = p->t0 > 0.0f;
                for (int64_t r = 0; r < nrows; ++r) {
                    int32_t &k0 = p->onfly_meta[(size_t)2 * r], &k1 = p->onfly_meta[(size_t)2 * r + 1];
                    const int32_t h0 = hi_meta[(size_t)2 * r], h1 = hi_meta[(size_t)2 * r + 1];
                    const int32_t a1 = k1 < 0 ? -1 : (k1 & 0x3FFFFFFF), b1 = h1 < 0 ? -1 : (h1 & 0x3FFFFFFF);
                    const bool va = a1 >= k0, vb = b1 >= h0;                 // any valid pixel at the low / high speed
                    const bool alla = va && (k1 >> 30 & 1), allb = vb && (h1 >> 30 & 1);
                    if (!vb && !early) { k0 = INT32_MAX; k1 = -1; continue; }   // beyond the record at every speed
                    int32_t lo = vb ? h0 : INT32_MAX, hi = va ? a1 : -1;
                    if (va) lo = std::min(lo, k0);
                    if (vb) hi = std::max(hi, b1);
                    if (!alla) hi = kend;
                    if (!allb && early) lo = 0;
                    if (hi < lo) { k0 = INT32_MAX; k1 = -1; continue; }
                    k0 = lo;
                    k1 = hi | (alla && allb ? 1 << 30 : 0);
                }
            }
        }
        plan_free(p, &mbuf);
        if (le || e != cudaSuccess) { p->onfly_meta.clear(); return cuda_fail(p, le ? le : (int)e, "conventional BP row ranges"); }
        p->onfly_c0 = c0;
        p->onfly_c0_hi = c0_hi;
        p->onfly_d2_in_range = bad == 0;
        needed_samples(p->onfly_meta, p->dims.nt, &p->onfly_lo, &p->onfly_hi);
        // work lists of the previous c0 are stale
        for (size_t q = 0; q < p->schedules.size();) {
            if (p->schedules[q].cfg.onfly) {
                plan_free(p, &p->schedules[q].buf);
                p->schedules.erase(p->schedules.begin() + (long)q);
            } else {
                ++q;
            }
        }
    }
    // the gather may use the written-out square root and skip "- t0" (gather.cu, onfly_u_fast2d): bit-identical there
    out->fast2d = p->grid.ndim == 2 && p->t0 == 0.0f && p->onfly_d2_in_range && !p->env.no_fast_delays;
    return PAT_OK;
}

}  // namespace

PatLayout pat_layout(const PatDims &d) {
    PatLayout L;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
    L.tau = take((size_t)d.ntiles * d.nsens * kTilePix * sizeof(float));
    L.meta = take((size_t)d.ntiles * d.nsens * 2 * sizeof(int32_t));
    const int bp = pat_frames_per_group(d.max_batch);
    const size_t padded = (size_t)(d.max_batch + bp - 1) / bp * bp;
    L.bd = take(padded * d.nsens * ((d.nt + 31) / 32 * 32) * sizeof(float));
    L.bd2 = take(padded * d.nsens * ((d.nt + 31) / 32 * 32) * sizeof(float));
    L.bd3 = take(padded * d.nsens * ((d.nt + 31) / 32 * 32) * sizeof(float));
    L.sync = take(768);
    L.perm = take((size_t)d.ntiles * kTilePix * sizeof(int32_t));
    L.traces = take((size_t)d.max_batch * d.nsens * d.nt * sizeof(float));
    L.traces2 = take((size_t)d.max_batch * d.nsens * d.nt * sizeof(float));
    L.images = take((size_t)d.max_batch * d.npix * sizeof(float));
    int64_t rows = (int64_t)((32u << 20) / ((size_t)d.npix * sizeof(float)));
    rows = std::max<int64_t>(1, std::min<int64_t>(rows, d.nsens));
    L.stage_rows = rows;
    L.tau_stage = take((size_t)rows * d.npix * sizeof(float));
    L.total = off;
    return L;
}

extern "C" size_t pat_plan_workspace_bytes(const pat_grid *grid, int32_t nsens, int64_t npix,
                                           int32_t nt, int32_t max_batch) {
    if (!dims_ok(grid, nsens, npix, nt, max_batch)) return 0;
    PatDims d;
    d.nsens = nsens; d.npix = npix; d.nt = nt; d.max_batch = max_batch;
    d.ntiles = (npix + kTilePix - 1) / kTilePix;
    return pat_layout(d).total;
}

// The order of the ROI pixels in the tile-major table (host only): slot -> ROI position, padded with -1 to whole tiles.
// May throw std::bad_alloc.
static std::vector<int32_t> build_pixel_order(const pat_grid *grid, const int64_t *roi_index, int64_t npix, bool plain_morton) {
    const int64_t ntiles = (npix + kTilePix - 1) / kTilePix;
    std::vector<int32_t> perm;
    {
        // spatially compact pixel order: sort ROI positions by the Morton key of their node
        std::vector<uint64_t> key((size_t)npix);
        const int64_t n0 = grid->n[0], n1 = grid->n[1];
        for (int64_t j = 0; j < npix; ++j) {
            const int64_t q = roi_index ? roi_index[j] : j;
            const uint32_t ix = (uint32_t)(q % n0), iy = (uint32_t)((q / n0) % n1), iz = (uint32_t)(q / (n0 * n1));
            key[j] = grid->ndim == 2 ? (spread2(ix) | (spread2(iy) << 1))
                                     : (spread3(ix) | (spread3(iy) << 1) | (spread3(iz) << 2));
        }
        perm.assign((size_t)ntiles * kTilePix, -1);
        std::iota(perm.begin(), perm.begin() + npix, 0);
        std::sort(perm.begin(), perm.begin() + npix,
                  [&](int32_t a, int32_t b) { return key[a] < key[b] || (key[a] == key[b] && a < b); });
        // A tile of the gather is 256 consecutive slots and a warp takes 32 of them.  Plain Morton order is compact
        // only where the region covers whole, ALIGNED blocks of the Morton grid: a disk (or a cube at an odd offset)
        // cuts blocks, everything behind the first partial block is shifted, and a warp or a tile then straddles
        // blocks that are neighbours on the Z-curve but not in space (configs[1]: 30 % of the warp rows span >= 32
        // samples -- bank conflicts in the blocked trace layout -- and a tile's window is 90 samples on average, 268
        // at the 99th percentile).  So the order is made by recursive coordinate bisection instead: split the pixel
        // set at a multiple of 256 across the longest axis of its bounding box until the parts are tiles, then every
        // tile the same way in halves down to groups of 8 (warps, half-warps and quarter-warps all compact; Morton order inside).  configs[1]: warp rows
        // spanning >= 32 samples 0.1 %, windows 64 samples on average, 89 at the 99th percentile, 94 at most.
        if (!plain_morton && npix > 32) {
            const int nd = grid->ndim;
            std::vector<int32_t> cx((size_t)npix), cy((size_t)npix), cz((size_t)npix);
            for (int64_t j = 0; j < npix; ++j) {
                const int64_t q = roi_index ? roi_index[j] : j;
                cx[(size_t)j] = (int32_t)(q % n0); cy[(size_t)j] = (int32_t)((q / n0) % n1); cz[(size_t)j] = (int32_t)(q / (n0 * n1));
            }
            // iterative bisection of perm[lo, hi) into parts of `unit` slots (the last part may be shorter)
            auto bisect = [&](int64_t lo0, int64_t hi0, int64_t unit) {
                std::vector<std::pair<int64_t, int64_t>> todo{{lo0, hi0}};
                while (!todo.empty()) {
                    const auto [lo, hi] = todo.back();
                    todo.pop_back();
                    if (hi - lo <= unit) continue;
                    int32_t mn[3] = {INT32_MAX, INT32_MAX, INT32_MAX}, mx[3] = {INT32_MIN, INT32_MIN, INT32_MIN};
                    for (int64_t q = lo; q < hi; ++q) {
                        const size_t a = (size_t)perm[(size_t)q];
                        const int32_t c[3] = {cx[a], cy[a], cz[a]};
                        for (int dd = 0; dd < nd; ++dd) { mn[dd] = std::min(mn[dd], c[dd]); mx[dd] = std::max(mx[dd], c[dd]); }
                    }
                    int ax = 0;
                    for (int dd = 1; dd < nd; ++dd) if (mx[dd] - mn[dd] > mx[ax] - mn[ax]) ax = dd;
                    const std::vector<int32_t> &co = ax == 0 ? cx : ax == 1 ? cy : cz;
                    const int64_t units = (hi - lo + unit - 1) / unit, cut = lo + units / 2 * unit;
                    std::nth_element(perm.begin() + lo, perm.begin() + cut, perm.begin() + hi, [&](int32_t a, int32_t b) {
                        return co[(size_t)a] < co[(size_t)b] || (co[(size_t)a] == co[(size_t)b] && key[(size_t)a] < key[(size_t)b]);
                    });
                    todo.push_back({lo, cut});
                    todo.push_back({cut, hi});
                }
            };
            bisect(0, npix, kTilePix);
            for (int64_t t0 = 0; t0 < npix; t0 += kTilePix) {
                const int64_t t1 = std::min<int64_t>(npix, t0 + kTilePix);
                bisect(t0, t1, 8);       // halves all the way down: 128, 64, 32 (a warp), 16 (a half-warp: 64-bit loads), 8
                for (int64_t w0 = t0; w0 < t1; w0 += 8)
                    std::sort(perm.begin() + w0, perm.begin() + std::min<int64_t>(t1, w0 + 8),
                              [&](int32_t a, int32_t b) { return key[(size_t)a] < key[(size_t)b]; });
            }
            // tiles in the Morton order of their first pixel: consecutive tiles (consecutive CTAs' shares) stay neighbours
            const int64_t nt_full = (npix + kTilePix - 1) / kTilePix;
            std::vector<int64_t> tord((size_t)nt_full);
            std::iota(tord.begin(), tord.end(), 0);
            auto tile_key = [&](int64_t t) {
                uint64_t m = ~0ull;
                for (int64_t q = t * kTilePix; q < std::min<int64_t>(npix, (t + 1) * kTilePix); ++q) m = std::min(m, key[(size_t)perm[(size_t)q]]);
                return m;
            };
            std::vector<uint64_t> tk((size_t)nt_full);
            for (int64_t t = 0; t < nt_full; ++t) tk[(size_t)t] = tile_key(t);
            // the short last tile stays last (its padding lanes end the slot array)
            std::sort(tord.begin(), tord.end() - ((npix % kTilePix) ? 1 : 0), [&](int64_t a, int64_t b) { return tk[(size_t)a] < tk[(size_t)b]; });
            std::vector<int32_t> tmp(perm.begin(), perm.begin() + npix);
            int64_t w = 0;
            for (int64_t t : tord)
                for (int64_t q = t * kTilePix; q < std::min<int64_t>(npix, (t + 1) * kTilePix); ++q) perm[(size_t)w++] = tmp[(size_t)q];
        }
    }
    return perm;
}

extern "C" pat_status pat_plan_create(pat_plan **out, const pat_grid *grid, const float *c_map,
                                      const float *sensor_xyz, int32_t nsens,
                                      const int64_t *roi_index, int64_t npix,
                                      int32_t nt, float fs, float t0,
                                      int32_t weighting, int32_t max_batch,
                                      void *workspace, size_t workspace_bytes) {
    // ---- argument checks: all of them run before the first CUDA call ---------------------
    if (!out) return fail(nullptr, PAT_ERR_INVALID_ARG, "out is NULL");
    if (!grid) return fail(nullptr, PAT_ERR_INVALID_ARG, "grid is NULL");
    if (!dims_ok(grid, nsens, npix, nt, max_batch))
        return fail(nullptr, PAT_ERR_INVALID_ARG, "bad sizes (ndim, n, h, nsens, npix, nt or max_batch)");
    if (!(fs > 0.0f) || !std::isfinite(fs) || !std::isfinite(t0))
        return fail(nullptr, PAT_ERR_INVALID_ARG, "fs must be finite and > 0, t0 finite");
    if (weighting < 0 || weighting > PAT_W_UBP_EXACT) return fail(nullptr, PAT_ERR_INVALID_ARG, "unknown weighting");
    int64_t N = 1;
    for (int d = 0; d < grid->ndim; ++d) N *= grid->n[d];
    if (!roi_index && npix != N)
        return fail(nullptr, PAT_ERR_INVALID_ARG, "roi_index NULL requires npix == number of nodes");
    if (roi_index)
        for (int64_t j = 0; j < npix; ++j) {
            if (roi_index[j] < 0 || roi_index[j] >= N || (j > 0 && roi_index[j] <= roi_index[j - 1]))
                return fail(nullptr, PAT_ERR_INVALID_ARG, "roi_index must be strictly ascending and inside the grid");
        }
    if (c_map)
        for (int64_t q = 0; q < N; ++q)
            if (!(c_map[q] > 0.0f) || !std::isfinite(c_map[q]))
                return fail(nullptr, PAT_ERR_INVALID_ARG, "c_map entries must be finite and > 0");
    if (sensor_xyz)
        for (int64_t q = 0; q < (int64_t)nsens * 3; ++q)
            if (!std::isfinite(sensor_xyz[q]))
                return fail(nullptr, PAT_ERR_INVALID_ARG, "sensor_xyz must be finite");
    if (!workspace) return fail(nullptr, PAT_ERR_INVALID_ARG, "workspace is NULL");
    if (((uintptr_t)workspace & 255u) != 0)
        return fail(nullptr, PAT_ERR_INVALID_ARG, "workspace must be 256-byte aligned");

    pat_plan *p = new (std::nothrow) pat_plan();
    if (!p) return fail(nullptr, PAT_ERR_NOMEM, "host allocation failed");
    p->dims.nsens = nsens; p->dims.npix = npix; p->dims.nt = nt; p->dims.max_batch = max_batch;
    p->dims.ntiles = (npix + kTilePix - 1) / kTilePix;
    p->lay = pat_layout(p->dims);
    if (workspace_bytes < p->lay.total) {
        delete p;
        return fail(nullptr, PAT_ERR_INVALID_ARG, "workspace smaller than pat_plan_workspace_bytes");
    }
    p->grid = *grid;
    if (grid->ndim == 2) { p->grid.n[2] = 1; p->grid.origin[2] = 0.0f; }
    p->fs = fs; p->t0 = t0; p->weighting = weighting;
    p->nt4 = (nt + 3) / 4 * 4;
    p->exact = weighting == PAT_W_PAPER_EXACT || weighting == PAT_W_UBP_EXACT;
    p->wp = (weighting == PAT_W_UBP || weighting == PAT_W_UBP_EXACT) ? 2.0f : 1.0f;
    p->wd = weighting == PAT_W_DELAY_SUM ? 0.0f : p->wp;
    p->ws = (char *)workspace;
    const char *env = std::getenv("PAT_NO_PDL");
    p->use_pdl = !(env && env[0] == '1');
    {   // tuning / diagnostic knobs: read here, once (PatTune)
        auto env_int = [](const char *n, int dflt) { const char *v = std::getenv(n); return v ? std::atoi(v) : dflt; };
        p->env.wr = env_int("PAT_WR", 0); p->env.R = env_int("PAT_R", 0); p->env.stages = env_int("PAT_STAGES", 0);
        p->env.cap = env_int("PAT_CAP", 0); p->env.budget_kb = env_int("PAT_BUDGET_KB", 0);
        p->env.chunk_cost = std::max(0, env_int("PAT_CHUNK_COST", 6));
        p->env.slow_cost = std::max(1, env_int("PAT_SLOW_COST", 5));
        p->env.debug = env_int("PAT_DEBUG", 0) == 1;
        p->env.chain_depth = env_int("PAT_CHAIN_DEPTH", 3);
        p->env.old_blocked_prepass = env_int("PAT_OLD_BLOCKED_PREPASS", 0) == 1;
        p->env.no_fast_delays = env_int("PAT_NO_FAST_DELAYS", 0) == 1;   // A/B: the generic delay arithmetic in the conventional BP
        if (const char *fn = std::getenv("PAT_SCHED_DUMP")) p->env.sched_dump = fn;
    }
    env = std::getenv("PAT_TRACE_FILE");                   // diagnostic: per-CTA timeline of the last gather launch
    p->trace_file = env && env[0];
    if (p->trace_file) p->trace_file_name = env;
    env = std::getenv("PAT_ENABLE_PROBES");                // measurement modes of pat_set_profiling (bench.py)
    p->probes = env && env[0] == '1';
    env = std::getenv("PAT_FULL_H2D");                     // A/B switch: always transfer whole traces
    p->window_h2d = !(env && env[0] == '1');
    env = std::getenv("PAT_FULL_PREPASS");                 // A/B switch: weight every sample of every trace
    p->window_prepass = !(env && env[0] == '1');

    std::vector<int32_t> perm;
    try {
        p->row_set.assign((size_t)nsens, 0);
        if (c_map) p->c_map.assign(c_map, c_map + N);
        if (sensor_xyz) p->sensors.assign(sensor_xyz, sensor_xyz + (int64_t)nsens * 3);
        if (roi_index) p->roi.assign(roi_index, roi_index + npix);
        perm = build_pixel_order(grid, roi_index, npix, std::getenv("PAT_PLAIN_MORTON") != nullptr);
    } catch (...) {
        delete p;
        return fail(nullptr, PAT_ERR_NOMEM, "host allocation failed");
    }

    // ---- device ---------------------------------------------------------------------------
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { delete p; return cuda_fail(nullptr, e, "cudaGetDevice (no usable CUDA device; there is no CPU fallback)"); }
    int major = 0, sms = 0;
    e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) { delete p; return cuda_fail(nullptr, e, "cudaDeviceGetAttribute"); }
    if (major != 10) {
        delete p;
        return fail(nullptr, PAT_ERR_UNSUPPORTED, "device is not sm_100 (Blackwell B200); no fallback path exists");
    }
    if (is_device_ptr(workspace) != 1) {
        delete p;
        return fail(nullptr, PAT_ERR_INVALID_ARG, "workspace is not device memory");
    }
    p->device = dev;
    p->num_sms = sms;
    p->alloc = pat_current_allocator();
    {
        int lo = 0, hi = 0;
        if (cudaDeviceGetStreamPriorityRange(&lo, &hi) == cudaSuccess) p->prio_high = hi; else cudaGetLastError();
    }
    p->host_perm = perm;
    e = cudaMemcpy(p->ws + p->lay.perm, perm.data(), perm.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemset(p->ws + p->lay.sync, 0, 768);
    if (e != cudaSuccess) { delete p; return cuda_fail(nullptr, e, "upload of the pixel permutation"); }
    if (!(std::getenv("PAT_NO_PIPE") && std::getenv("PAT_NO_PIPE")[0] == '1')) {
        cudaStream_t cs = nullptr;
        bool ok = cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking) == cudaSuccess;
        for (int q = 0; q < 2 && ok; ++q) {
            cudaEvent_t a = nullptr, b = nullptr;
            ok = cudaEventCreateWithFlags(&a, cudaEventDisableTiming) == cudaSuccess &&
                 cudaEventCreateWithFlags(&b, cudaEventDisableTiming) == cudaSuccess;
            p->ev_h2d[q] = a; p->ev_read[q] = b;
        }
        if (ok) p->copy_stream = cs;                   // otherwise host calls stay serial on the caller's stream
        else if (cs) cudaStreamDestroy(cs);
    }
    *out = p;
    return PAT_OK;
}

// Rows [sensor_begin, +count) of a row-major [count][npix] table (host or device) -> the tile-major table
// `dst_t`, every value mapped to fl32(fl32(v - t0) * fs) (fs = 1, t0 = 0: copied unchanged).
static pat_status upload_rows(pat_plan *p, const float *src, int32_t sensor_begin, int32_t count, float *dst_t,
                              float fs, float t0, void *stream) {
    const int on_dev = is_device_ptr(src);
    if (on_dev < 0) return fail(p, PAT_ERR_CUDA, "cudaPointerGetAttributes failed on the table rows");
    cudaStream_t st = (cudaStream_t)stream;
    PatLaunchCtx ctx{stream, p->num_sms, p->use_pdl};
    const int32_t *perm = (const int32_t *)(p->ws + p->lay.perm);
    const int64_t P = p->dims.npix;
    if (on_dev) {
        int e = pat_launch_retile(ctx, src, dst_t, perm, p->dims.nsens, P, p->dims.ntiles, sensor_begin, count, fs, t0);
        if (e) return cuda_fail(p, e, "retile launch");
        ++p->launches;
    } else {
        float *stage = (float *)(p->ws + p->lay.tau_stage);
        for (int32_t r = 0; r < count; r += (int32_t)p->lay.stage_rows) {
            const int32_t m = (int32_t)std::min<int64_t>(p->lay.stage_rows, count - r);
            cudaError_t e = cudaMemcpyAsync(stage, src + (int64_t)r * P, (size_t)m * P * sizeof(float),
                                            cudaMemcpyHostToDevice, st);
            if (e != cudaSuccess) return cuda_fail(p, e, "table H2D copy");
            int le = pat_launch_retile(ctx, stage, dst_t, perm, p->dims.nsens, P, p->dims.ntiles,
                                       sensor_begin + r, m, fs, t0);
            if (le) return cuda_fail(p, le, "retile launch");
            ++p->launches;
            // the staging buffer is reused by the next piece and the host rows are only
            // borrowed until return: wait for this piece.
            e = cudaStreamSynchronize(st);
            if (e != cudaSuccess) return cuda_fail(p, e, "table staging synchronise");
        }
    }
    return PAT_OK;
}

extern "C" pat_status pat_set_travel_times(pat_plan *p, const float *tau, int32_t sensor_begin,
                                           int32_t count, void *stream) {
    if (!p) return PAT_ERR_INVALID_ARG;
    if (pat_status ds = check_device(p)) return ds;
    if (!tau && count > 0) return fail(p, PAT_ERR_INVALID_ARG, "tau is NULL");
    if (sensor_begin < 0 || count < 0 || sensor_begin > p->dims.nsens - count)
        return fail(p, PAT_ERR_INVALID_ARG, "sensor range outside [0, nsens)");
    if (count == 0) return PAT_OK;
    pat_status us = upload_rows(p, tau, sensor_begin, count, (float *)(p->ws + p->lay.tau), p->fs, p->t0, stream);
    if (us != PAT_OK) return us;
    for (int32_t s = sensor_begin; s < sensor_begin + count; ++s)
        if (!p->row_set[s]) { p->row_set[s] = 1; ++p->rows_set; }
    p->meta_valid = false;
    drop_schedules(p);
    if (p->rows_set == p->dims.nsens) return finalize_table(p, stream);
    return PAT_OK;
}

static pat_status backproject_impl(pat_plan *p, const float *traces, float *images, int32_t nframes, void *stream,
                                   bool conventional, float c0, const float *sweep_c0 = nullptr, int32_t nsweep = 0);

extern "C" pat_status pat_backproject(pat_plan *p, const float *traces, float *images,
                                      int32_t nframes, void *stream) {
    return backproject_impl(p, traces, images, nframes, stream, false, 0.0f);
}

extern "C" pat_status pat_backproject_conventional(pat_plan *p, const float *traces, float *images,
                                                   int32_t nframes, float c0, void *stream) {
    if (!p) return PAT_ERR_INVALID_ARG;
    if (pat_status ds = check_device(p)) return ds;
    if (!(c0 > 0.0f) || !std::isfinite(c0)) return fail(p, PAT_ERR_INVALID_ARG, "c0 must be finite and > 0");
    if (p->sensors.empty()) return fail(p, PAT_ERR_BAD_STATE, "plan was created without sensor_xyz");
    return backproject_impl(p, traces, images, nframes, stream, true, c0);
}

extern "C" pat_status pat_backproject_conventional_sweep(pat_plan *p, const float *traces, float *images,
                                                         const float *c0, int32_t nc0, void *stream) {
    if (!p) return PAT_ERR_INVALID_ARG;
    if (!c0 || nc0 < 1 || nc0 > PAT_MAX_SWEEP) return fail(p, PAT_ERR_INVALID_ARG, "c0 is NULL or nc0 outside [1, PAT_MAX_SWEEP]");
    for (int32_t q = 0; q < nc0; ++q)
        if (!(c0[q] > 0.0f) || !std::isfinite(c0[q])) return fail(p, PAT_ERR_INVALID_ARG, "every c0 must be finite and > 0");
    if (p->sensors.empty()) return fail(p, PAT_ERR_BAD_STATE, "plan was created without sensor_xyz");
    if (p->exact) return fail(p, PAT_ERR_UNSUPPORTED, "the sweep is not available with the _EXACT weightings");
    if (p->d_w_t) return fail(p, PAT_ERR_UNSUPPORTED, "the sweep is not combined with pixel weights");
    return backproject_impl(p, traces, images, 1, stream, true, c0[0], c0, nc0);
}

static pat_status backproject_impl(pat_plan *p, const float *traces, float *images, int32_t nframes, void *stream,
                                   bool conventional, float c0, const float *sweep_c0, int32_t nsweep) {
    if (!p) return PAT_ERR_INVALID_ARG;
    const int32_t nimages = nsweep > 0 ? nsweep : nframes;      // a sweep: ONE frame of traces, one image per speed
    if (nframes < 0 || nframes > p->dims.max_batch)
        return fail(p, PAT_ERR_INVALID_ARG, "nframes outside [0, max_batch]");
    const int32_t nch = p->exact ? 2 * nframes : nframes;       // exact-time weightings: two channels per frame
    if (nch > p->dims.max_batch)
        return fail(p, PAT_ERR_INVALID_ARG, "the _EXACT weightings need nframes <= max_batch/2 (two channels per frame)");
    if (nframes == 0) return PAT_OK;
    if (!traces || !images) return fail(p, PAT_ERR_INVALID_ARG, "traces or images is NULL");
    if (!conventional && p->rows_set != p->dims.nsens)
        return fail(p, PAT_ERR_BAD_STATE, "pat_backproject before every tau row was set");
    const int td = is_device_ptr(traces), id = is_device_ptr(images);
    if (td < 0 || id < 0) return fail(p, PAT_ERR_CUDA, "cudaPointerGetAttributes failed");
    if (td != id) return fail(p, PAT_ERR_INVALID_ARG, "traces and images must both be host or both device");
    if (td && ((((uintptr_t)traces) | ((uintptr_t)images)) & 15u))
        return fail(p, PAT_ERR_INVALID_ARG, "device traces/images must be 16-byte aligned");
    if (nsweep > 0 && !td) return fail(p, PAT_ERR_UNSUPPORTED, "the sweep takes DEVICE buffers");

    cudaStream_t st = (cudaStream_t)stream;
    const PatDims &d = p->dims;
    const float *d_tr = traces;
    float *d_img = images;
    const int slot = (int)(p->host_calls & 1u);
    bool piped = false;
    PatOnfly onfly;
    if (conventional) {      // geometry + k-ranges for this c0 (first use: builds them, synchronous)
        float c_lo = c0, c_hi = c0;
        for (int32_t q = 0; q < nsweep; ++q) { c_lo = std::min(c_lo, sweep_c0[q]); c_hi = std::max(c_hi, sweep_c0[q]); }
        pat_status os = ensure_onfly(p, c_lo, c_hi, stream, &onfly);
        if (os != PAT_OK) return os;
        onfly.nsweep = nsweep;
        for (int32_t q = 0; q < nsweep; ++q) onfly.sweep_inv_c0[q] = 1.0f / sweep_c0[q];
    }
    if (!td) {
        d_tr = (const float *)(p->ws + (slot ? p->lay.traces2 : p->lay.traces));
        d_img = (float *)(p->ws + p->lay.images);
        const size_t tbytes = (size_t)nframes * d.nsens * d.nt * sizeof(float);
        // only the samples the table can touch cross the bus (PAPER.md:79 counts the transfers): one strided copy
        // of [lo, hi) of every trace when that is well below the whole record; the rest of the staging buffer is
        // never read by a valid pixel
        const int32_t lo = conventional ? p->onfly_lo : p->need_lo, hi = conventional ? p->onfly_hi : p->need_hi;
        const bool windowed = p->window_h2d && (int64_t)(hi - lo) * 5 <= (int64_t)d.nt * 4;
        auto h2d = [&](cudaStream_t s_) -> cudaError_t {
            if (!windowed) return cudaMemcpyAsync((void *)d_tr, traces, tbytes, cudaMemcpyHostToDevice, s_);
            if (hi <= lo) return cudaSuccess;
            return cudaMemcpy2DAsync((void *)(d_tr + lo), (size_t)d.nt * sizeof(float), traces + lo,
                                     (size_t)d.nt * sizeof(float), (size_t)(hi - lo) * sizeof(float),
                                     (size_t)nframes * d.nsens, cudaMemcpyHostToDevice, s_);
        };
        cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
        cudaStreamIsCapturing(st, &cap);
        piped = p->copy_stream && cap == cudaStreamCaptureStatusNone;
        cudaError_t e;
        if (piped) {
            // the copy runs on the plan's copy stream, i.e. under the kernels of the previous call; it may
            // overwrite this staging buffer once the pre-pass of the call before last has read it
            cudaStream_t cs = (cudaStream_t)p->copy_stream;
            e = p->host_calls >= 2 ? cudaStreamWaitEvent(cs, (cudaEvent_t)p->ev_read[slot], 0) : cudaSuccess;
            if (e == cudaSuccess) e = h2d(cs);
            if (e == cudaSuccess) e = cudaEventRecord((cudaEvent_t)p->ev_h2d[slot], cs);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(st, (cudaEvent_t)p->ev_h2d[slot], 0);
        } else {
            e = h2d(st);
        }
        if (e != cudaSuccess) return cuda_fail(p, e, "traces H2D copy");
        ++p->host_calls;
    }
    const int bp = pat_frames_per_group(nch);
    PatSchedule *sc = nullptr;
    {   // first use of this frame-count class after the table (or c0) changed: builds the work list (synchronous)
        pat_status ss = get_schedule(p, bp, conventional, &sc);
        if (ss != PAT_OK) return ss;
    }
    const bool prof = p->profiling == 1 && p->prof_events.size() < 3u * 65536u;
    PatLaunchCtx ctx{stream, p->num_sms, p->use_pdl && !prof};
    ctx.high_priority = p->prio_high;
    ctx.old_blocked_prepass = p->env.old_blocked_prepass;
    const size_t ibytes = (size_t)nimages * d.npix * sizeof(float);
    const bool do_gather = sc->grid_x > 0 && p->profiling != 3;
    const bool do_pre = p->profiling != 2;
    // launch chain (see the top of this file): only for device buffers inside a capture
    ChainPlan cp;
    if (ctx.use_pdl && td && p->profiling != 4)
        cp = chain_begin(st, traces, (size_t)nframes * d.nsens * d.nt * sizeof(float), images, ibytes, p->env.chain_depth);
    if (cp.chained && !do_gather) cp.chained = false;
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
    if (prof) {
        for (int q = 0; q < 3; ++q) {
            cudaError_t ee = cudaEventCreate(&ev[q]);
            if (ee != cudaSuccess) return cuda_fail(p, ee, "cudaEventCreate");
            p->prof_events.push_back(ev[q]);
        }
        cudaEventRecord(ev[0], st);
    }
    // consecutive calls rotate through the three b buffers and their counters
    const int slot_b = p->b_slot;
    p->b_slot = (p->b_slot + 1) % 3;
    float *bw = (float *)(p->ws + (slot_b == 0 ? p->lay.bd : slot_b == 1 ? p->lay.bd2 : p->lay.bd3));
    uint32_t *sync = (uint32_t *)(p->ws + p->lay.sync) + 64 * slot_b;
    const float t0fs = (float)((double)p->t0 * (double)p->fs);
    int e = 0;
    if (p->sync_dirty) {              // an earlier call failed between its two launches: counters may be non-zero
        cudaError_t ce = cudaMemsetAsync(p->ws + p->lay.sync, 0, 768, st);
        if (ce != cudaSuccess) return cuda_fail(p, ce, "counter reset");
        p->sync_dirty = false;
    }
    if (p->profiling == 4) {          // measurement: the step's footprint (table + b in, images out) as a plain stream
        e = pat_launch_stream_probe(ctx, p->ws + p->lay.tau, (int64_t)d.ntiles * kTilePix * d.nsens * 4,
                                    bw, (int64_t)nch * d.nsens * p->nt4 * 4, d_img, (int64_t)nframes * d.npix);
        if (e) return cuda_fail(p, e, "stream probe launch");
        ++p->launches;
        return PAT_OK;
    }
    if (do_gather && p->trace_file && !p->trace_dev && nframes <= 32) {   // diagnostic timeline (PAT_TRACE_FILE at create)
        if (plan_alloc(p, (size_t)(sc->grid_x + 1) * 8 * sizeof(unsigned long long), &p->trace_buf)) {
            p->trace_dev = (unsigned long long *)p->trace_buf.p;
            p->trace_ctas = sc->grid_x;
            cudaMemset(p->trace_dev, 0, (size_t)(sc->grid_x + 1) * 8 * sizeof(unsigned long long));
        } else {
            p->trace_dev = nullptr;
        }
    }
    if (p->trace_dev && p->trace_ctas == sc->grid_x) ctx.pre_trace = p->trace_dev + (size_t)sc->grid_x * 8;
    cudaGraphNode_t node_pre = nullptr, node_gather = nullptr;
    unsigned long long cid = 0;
    if (do_pre) {
        if (cp.chained) {             // P_j behind P_{j-1} and G_{j-3} only
            cudaError_t ce = set_capture_deps(st, cp.pre_dep, cp.bound_dep, nullptr);
            if (ce != cudaSuccess) return cuda_fail(p, ce, "capture dependencies (pre-pass)");
        }
        e = pat_launch_prepass(ctx, d_tr, bw, d_img, d.nsens, d.nt, p->nt4, nframes, bp, d.npix, p->wp, p->wd, t0fs, p->exact,
                               p->window_prepass ? (conventional ? p->onfly_lo : p->need_lo) : 0,
                               p->window_prepass ? (conventional ? p->onfly_hi : p->need_hi) : INT32_MAX,
                               do_gather && !cp.chained ? sync : nullptr,    // chained: a full edge orders P before G
                               (int64_t)nimages * d.npix);
        if (e) return cuda_fail(p, e, "pre-pass launch");
        ++p->launches;
        if (cp.capture_id) capture_deps(st, &cid, &node_pre);
    }
    if (prof) cudaEventRecord(ev[1], st);
    if (piped) cudaEventRecord((cudaEvent_t)p->ev_read[slot], st);        // the staged traces have been consumed
    if (do_gather) {
        if (cp.chained) {             // G_j: full edges from P_j (and G_{j-3}), programmatic edge from G_{j-1}
            cudaError_t ce = set_capture_deps(st, node_pre, do_pre ? nullptr : cp.bound_dep, cp.prev_gather);
            if (ce != cudaSuccess) { p->sync_dirty = do_pre; return cuda_fail(p, ce, "capture dependencies (gather)"); }
            ctx.use_pdl = false;      // the edges are explicit: no launch attribute
            ++p->chained;
        }
        e = pat_launch_gather(ctx, sc->cfg, (const float *)(p->ws + p->lay.tau), bw, sc->d_sched, sc->d_first, sc->d_cta_chunk,
                              sc->grid_x, p->d_perm_masked ? p->d_perm_masked : (const int32_t *)(p->ws + p->lay.perm),
                              d_img, d.nsens, d.npix, d.nt,
                              p->nt4, nframes, p->trace_ctas == sc->grid_x ? p->trace_dev : nullptr,
                              conventional ? &onfly : nullptr, t0fs, p->d_w_t,
                              do_pre && !cp.chained ? sync : nullptr);
        if (e) { p->sync_dirty = do_pre; return cuda_fail(p, e, "gather launch"); }
        ++p->launches;
        if (cp.capture_id) capture_deps(st, &cid, &node_gather);
    }
    if (cp.capture_id && td) chain_commit(cp, do_pre ? node_pre : node_gather, node_gather, images, ibytes);
    if (prof) cudaEventRecord(ev[2], st);
    if (!td) {
        cudaError_t ce = cudaMemcpyAsync(images, d_img, (size_t)nframes * d.npix * sizeof(float),
                                         cudaMemcpyDeviceToHost, st);
        if (ce != cudaSuccess) return cuda_fail(p, ce, "images D2H copy");
    }
    return PAT_OK;
}

static void drop_events(pat_plan *p) {
    for (void *e : p->prof_events) cudaEventDestroy((cudaEvent_t)e);
    p->prof_events.clear();
}

extern "C" pat_status pat_destroy(pat_plan *p) {
    if (p && p->trace_dev) {                   // PAT_TRACE_FILE: dump the per-CTA timeline of the last launch
        std::vector<unsigned long long> h((size_t)(p->trace_ctas + 1) * 8);
        cudaDeviceSynchronize();
        if (cudaMemcpy(h.data(), p->trace_dev, h.size() * 8, cudaMemcpyDeviceToHost) == cudaSuccess)
            if (p->trace_file) {                   // one file per plan: <name>.<k>, k counting the plans destroyed so far
                static std::atomic<int> serial{0};
                const std::string fn = p->trace_file_name + "." + std::to_string(serial.fetch_add(1));
                if (FILE *f = std::fopen(fn.c_str(), "wb")) { std::fwrite(h.data(), 8, h.size(), f); std::fclose(f); }
            }
        plan_free(p, &p->trace_buf);
    }
    if (p) {
        drop_events(p); drop_schedules(p);
        plan_free(p, &p->mask_buf);
        plan_free(p, &p->w_buf);
        plan_free(p, &p->onfly_buf);
        if (p->copy_stream) { cudaStreamSynchronize((cudaStream_t)p->copy_stream); cudaStreamDestroy((cudaStream_t)p->copy_stream); }
        for (int q = 0; q < 2; ++q) {
            if (p->ev_h2d[q]) cudaEventDestroy((cudaEvent_t)p->ev_h2d[q]);
            if (p->ev_read[q]) cudaEventDestroy((cudaEvent_t)p->ev_read[q]);
        }
    }
    delete p;
    return PAT_OK;
}

extern "C" pat_status pat_set_profiling(pat_plan *p, int32_t enable) {
    if (!p) return PAT_ERR_INVALID_ARG;
    if (enable < 0 || enable > 4) return fail(p, PAT_ERR_INVALID_ARG, "profiling mode must be 0..4");
    if (enable >= 2 && !p->probes)
        return fail(p, PAT_ERR_UNSUPPORTED, "modes 2-4 leave garbage images: measurement only, plan must be created with PAT_ENABLE_PROBES=1");
    p->profiling = enable;
    return PAT_OK;
}

extern "C" pat_status pat_get_profile(pat_plan *p, int32_t reset, int64_t *calls, double *prepass_ms,
                                      double *gather_ms) {
    if (!p) return PAT_ERR_INVALID_ARG;
    double a = 0.0, b = 0.0;
    const size_t n = p->prof_events.size() / 3;
    for (size_t q = 0; q < n; ++q) {
        cudaEvent_t *ev = (cudaEvent_t *)&p->prof_events[3 * q];
        cudaError_t e = cudaEventSynchronize(ev[2]);
        float m0 = 0.f, m1 = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&m0, ev[0], ev[1]);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&m1, ev[1], ev[2]);
        if (e != cudaSuccess) return cuda_fail(p, e, "profile events");
        a += m0; b += m1;
    }
    if (calls) *calls = (int64_t)n;
    if (prepass_ms) *prepass_ms = a;
    if (gather_ms) *gather_ms = b;
    if (reset) drop_events(p);
    return PAT_OK;
}

extern "C" const char *pat_last_error(const pat_plan *p) {
    return p ? p->err.c_str() : g_create_error.c_str();
}

extern "C" int64_t pat_kernel_launches(const pat_plan *p) { return p ? p->launches : 0; }

extern "C" int64_t pat_chained_calls(const pat_plan *p) { return p ? p->chained : 0; }

extern "C" pat_status pat_get_stats(const pat_plan *p, pat_stats *out) {
    if (!p || !out) return PAT_ERR_INVALID_ARG;
    std::memset(out, 0, sizeof(*out));
    out->workspace_bytes = (int64_t)p->lay.total;
    out->provider_bytes = p->dev_bytes;
    out->provider_bytes_peak = p->dev_bytes_peak;
    for (const PatSchedule &sc : p->schedules) out->work_list_bytes += (int64_t)sc.buf.bytes;
    out->work_lists = p->sched_builds;
    out->work_list_build_seconds = p->sched_build_seconds;
    out->kernel_launches = p->launches;
    out->chained_calls = p->chained;
    return PAT_OK;
}

extern "C" pat_status pat_get_trace_window(const pat_plan *p, int32_t *first, int32_t *count) {
    if (!p || !first || !count) return PAT_ERR_INVALID_ARG;
    if (!p->meta_valid) return PAT_ERR_BAD_STATE;
    const int32_t lo = p->need_lo, hi = p->need_hi;
    const bool windowed = p->window_h2d && (int64_t)(hi - lo) * 5 <= (int64_t)p->dims.nt * 4;
    *first = windowed ? lo : 0;
    *count = windowed ? hi - lo : p->dims.nt;
    return PAT_OK;
}

extern "C" pat_status pat_set_gather_tuning(pat_plan *p, int32_t wr, int32_t rows, int32_t stages) {
    if (!p) return PAT_ERR_INVALID_ARG;
    if (wr < 0 || rows < 0 || stages < 0 || rows > 30 || stages > 8 || (wr && (wr < 8 || wr > 4096 || (wr & (wr - 1)))))
        return fail(p, PAT_ERR_INVALID_ARG, "wr: 0 or a power of two in [8, 4096]; rows: 0..30; stages: 0..8");
    if (stages == 1) return fail(p, PAT_ERR_INVALID_ARG, "stages must be 0 or >= 2");
    p->tune_wr = wr; p->tune_R = rows; p->tune_stages = stages;
    drop_schedules(p);
    return PAT_OK;
}

extern "C" pat_status pat_compute_travel_times(pat_plan *p, int32_t order, int32_t nthreads, void *stream) {
    if (!p) return PAT_ERR_INVALID_ARG;
    if (p->c_map.empty() || p->sensors.empty())
        return fail(p, PAT_ERR_BAD_STATE, "plan was created without c_map / sensor_xyz");
    const int64_t P = p->dims.npix;
    int64_t rows = std::max<int64_t>(1, std::min<int64_t>(p->dims.nsens, (int64_t)(256u << 20) / (P * 4)));
    std::vector<float> buf;
    try { buf.resize((size_t)rows * P); } catch (...) { return fail(p, PAT_ERR_NOMEM, "host allocation failed"); }
    for (int32_t s = 0; s < p->dims.nsens; s += (int32_t)rows) {
        const int32_t m = (int32_t)std::min<int64_t>(rows, p->dims.nsens - s);
        pat_status st = pat_fmm_travel_times(&p->grid, p->c_map.data(), p->sensors.data(), p->dims.nsens,
                                             p->roi.empty() ? nullptr : p->roi.data(), P, s, m, order,
                                             buf.data(), nthreads);
        if (st != PAT_OK) return fail(p, st, "pat_fmm_travel_times failed (sensor outside the grid?)");
        st = pat_set_travel_times(p, buf.data(), s, m, stream);
        if (st != PAT_OK) return st;
    }
    return PAT_OK;
}

extern "C" pat_status pat_compute_travel_times_gpu(pat_plan *p, int32_t max_rounds, int32_t *rounds_out,
                                                   void *stream) {
    if (!p) return PAT_ERR_INVALID_ARG;
    if (pat_status ds = check_device(p)) return ds;
    if (p->c_map.empty() || p->sensors.empty())
        return fail(p, PAT_ERR_BAD_STATE, "plan was created without c_map / sensor_xyz");
    float *stage = (float *)(p->ws + p->lay.tau_stage);
    const int32_t rows = (int32_t)std::max<int64_t>(1, p->lay.stage_rows);
    int32_t worst = 0;
    for (int32_t s = 0; s < p->dims.nsens; s += rows) {
        const int32_t m = std::min(rows, p->dims.nsens - s);
        int32_t r = 0;
        pat_status st = pat_eikonal_travel_times_device(&p->grid, p->c_map.data(), p->sensors.data(), p->dims.nsens,
                                                        p->roi.empty() ? nullptr : p->roi.data(), p->dims.npix, s, m,
                                                        stage, max_rounds, &r, stream);
        if (st != PAT_OK) return fail(p, st, "pat_eikonal_travel_times_device failed (sensor outside the grid, or no convergence)");
        worst = std::max(worst, r);
        st = pat_set_travel_times(p, stage, s, m, stream);
        if (st != PAT_OK) return st;
        if (cudaStreamSynchronize((cudaStream_t)stream) != cudaSuccess) return fail(p, PAT_ERR_CUDA, "synchronise");
    }
    if (rounds_out) *rounds_out = worst;
    return PAT_OK;
}

// The weight table exists from the first call on (all ones = no effect) and is library-owned.
static pat_status ensure_weight_table(pat_plan *p, void *stream) {
    if (p->exact)
        return fail(p, PAT_ERR_UNSUPPORTED, "pixel weights are not available with the _EXACT weightings");
    if (p->d_w_t) return PAT_OK;
    cudaError_t e = cudaDeviceSynchronize();            // no launch may still use the unweighted work lists
    if (e != cudaSuccess) return cuda_fail(p, e, "synchronise");
    const int64_t n = p->dims.ntiles * (int64_t)p->dims.nsens * kTilePix;
    if (!plan_alloc(p, (size_t)n * sizeof(float), &p->w_buf))
        return fail(p, PAT_ERR_NOMEM, "weight table: the device-memory provider returned nothing");
    p->d_w_t = (float *)p->w_buf.p;
    PatLaunchCtx ctx{stream, p->num_sms, false};
    int le = pat_launch_fill(ctx, p->d_w_t, n, 1.0f);
    if (le) { plan_free(p, &p->w_buf); p->d_w_t = nullptr; return cuda_fail(p, le, "weight table fill"); }
    ++p->launches;
    drop_schedules(p);                                  // the stages now hold weight rows as well
    return PAT_OK;
}

extern "C" pat_status pat_set_pixel_weights(pat_plan *p, const float *w, int32_t sensor_begin, int32_t count,
                                            void *stream) {
    if (!p) return PAT_ERR_INVALID_ARG;
    if (pat_status ds = check_device(p)) return ds;
    if (!w) {                                           // remove the weights
        if (count != 0) return fail(p, PAT_ERR_INVALID_ARG, "w is NULL");
        if (p->d_w_t) {
            cudaError_t e = cudaDeviceSynchronize();
            if (e != cudaSuccess) return cuda_fail(p, e, "synchronise");
            plan_free(p, &p->w_buf);
            p->d_w_t = nullptr;
            drop_schedules(p);
        }
        return PAT_OK;
    }
    if (sensor_begin < 0 || count < 0 || sensor_begin > p->dims.nsens - count)
        return fail(p, PAT_ERR_INVALID_ARG, "sensor range outside [0, nsens)");
    pat_status st = ensure_weight_table(p, stream);
    if (st != PAT_OK || count == 0) return st;
    return upload_rows(p, w, sensor_begin, count, p->d_w_t, 1.0f, 0.0f, stream);
}

extern "C" pat_status pat_compute_solid_angle_weights(pat_plan *p, const float *normals, void *stream) {
    if (!p) return PAT_ERR_INVALID_ARG;
    if (pat_status ds = check_device(p)) return ds;
    if (!normals) return fail(p, PAT_ERR_INVALID_ARG, "normals is NULL");
    if (p->sensors.empty()) return fail(p, PAT_ERR_BAD_STATE, "plan was created without sensor_xyz");
    const int32_t S = p->dims.nsens;
    for (int64_t q = 0; q < (int64_t)S * 3; ++q)
        if (!std::isfinite(normals[q])) return fail(p, PAT_ERR_INVALID_ARG, "normals must be finite");
    pat_status st = ensure_weight_table(p, stream);
    if (st != PAT_OK) return st;
    // node coordinates of every tile slot in double: x_d = origin_d + i_d * h from the fp32 grid data
    const int64_t slots = p->dims.ntiles * kTilePix;
    std::vector<double> pix;
    try { pix.assign((size_t)slots * 3, 0.0); } catch (...) { return fail(p, PAT_ERR_NOMEM, "host allocation failed"); }
    const int64_t n0 = p->grid.n[0], n1 = p->grid.n[1];
    for (int64_t sl = 0; sl < slots; ++sl) {
        int32_t pos = p->host_perm[(size_t)sl];
        if (pos < 0) pos = p->host_perm[(size_t)(sl / kTilePix * kTilePix)];          // padding: the tile's first pixel
        const int64_t q = p->roi.empty() ? pos : p->roi[(size_t)pos];
        const int64_t id[3] = {q % n0, (q / n0) % n1, q / (n0 * n1)};
        for (int dd = 0; dd < p->grid.ndim; ++dd)
            pix[(size_t)dd * slots + sl] = (double)p->grid.origin[dd] + (double)id[dd] * (double)p->grid.h;
    }
    cudaStream_t cs = (cudaStream_t)stream;
    PatDevBuf tmp;                                      // node coordinates, then sensors, then normals
    const size_t pix_bytes = align_up(pix.size() * sizeof(double), 256);
    if (!plan_alloc(p, pix_bytes + (size_t)S * 6 * sizeof(float), &tmp))
        return fail(p, PAT_ERR_NOMEM, "solid-angle scratch: the device-memory provider returned nothing");
    double *d_pix = (double *)tmp.p;
    float *d_sn = (float *)((char *)tmp.p + pix_bytes);
    cudaError_t e = cudaSuccess;
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_pix, pix.data(), pix.size() * sizeof(double), cudaMemcpyHostToDevice, cs);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_sn, p->sensors.data(), (size_t)S * 3 * sizeof(float), cudaMemcpyHostToDevice, cs);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_sn + (size_t)S * 3, normals, (size_t)S * 3 * sizeof(float), cudaMemcpyHostToDevice, cs);
    int le = 0;
    if (e == cudaSuccess) {
        PatLaunchCtx ctx{stream, p->num_sms, false};
        le = pat_launch_solid_angle(ctx, d_pix, slots, d_sn, d_sn + (size_t)S * 3, S, p->grid.ndim, p->d_w_t);
        ++p->launches;
    }
    if (e == cudaSuccess && !le) e = cudaStreamSynchronize(cs);       // the host arrays are only borrowed
    else cudaStreamSynchronize(cs);
    plan_free(p, &tmp);
    if (le) return cuda_fail(p, le, "solid-angle launch");
    if (e != cudaSuccess) return cuda_fail(p, e, "solid-angle weights");
    return PAT_OK;
}

extern "C" pat_status pat_set_roi_mask(pat_plan *p, const uint8_t *mask) {
    if (!p) return PAT_ERR_INVALID_ARG;
    if (pat_status ds = check_device(p)) return ds;
    cudaError_t e = cudaDeviceSynchronize();            // no launch may still read the old permutation / lists
    if (e != cudaSuccess) return cuda_fail(p, e, "synchronise");
    drop_schedules(p);
    if (!mask) {
        p->tile_active.clear();
        plan_free(p, &p->mask_buf);
        p->d_perm_masked = nullptr;
        return PAT_OK;
    }
    const int64_t slots = p->dims.ntiles * kTilePix;
    std::vector<int32_t> perm;
    try {
        perm = p->host_perm;
        p->tile_active.assign((size_t)p->dims.ntiles, 0);
    } catch (...) { return fail(p, PAT_ERR_NOMEM, "host allocation failed"); }
    for (int64_t sl = 0; sl < slots; ++sl) {
        const int32_t pos = perm[(size_t)sl];
        if (pos < 0) continue;
        if (mask[pos]) p->tile_active[(size_t)(sl / kTilePix)] = 1;
        else perm[(size_t)sl] = -1;
    }
    if (!p->d_perm_masked) {
        if (!plan_alloc(p, (size_t)slots * sizeof(int32_t), &p->mask_buf)) {
            p->tile_active.clear();
            return fail(p, PAT_ERR_NOMEM, "roi mask: the device-memory provider returned nothing");
        }
        p->d_perm_masked = (int32_t *)p->mask_buf.p;
    }
    e = cudaMemcpy(p->d_perm_masked, perm.data(), (size_t)slots * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return cuda_fail(p, e, "roi mask upload");
    return PAT_OK;
}

// Host only (no CUDA call): the slot order pat_plan_create would use for this region -- for tests of the order's
// properties and for callers that want to lay out their own per-pixel data tile-major.
extern "C" pat_status pat_pixel_order(const pat_grid *grid, const int64_t *roi_index, int64_t npix, int32_t plain_morton,
                                      int32_t *perm_out) {
    if (!grid || !perm_out || npix <= 0 || npix > (int64_t)INT32_MAX) return PAT_ERR_INVALID_ARG;
    if (grid->ndim != 2 && grid->ndim != 3) return PAT_ERR_INVALID_ARG;
    int64_t N = 1;
    for (int dd = 0; dd < grid->ndim; ++dd) { if (grid->n[dd] < 1) return PAT_ERR_INVALID_ARG; N *= grid->n[dd]; }
    if (!roi_index && npix != N) return PAT_ERR_INVALID_ARG;
    if (roi_index)
        for (int64_t j = 0; j < npix; ++j)
            if (roi_index[j] < 0 || roi_index[j] >= N) return PAT_ERR_INVALID_ARG;
    try {
        const std::vector<int32_t> perm = build_pixel_order(grid, roi_index, npix, plain_morton != 0);
        std::copy(perm.begin(), perm.end(), perm_out);
    } catch (...) { return PAT_ERR_NOMEM; }
    return PAT_OK;
}
