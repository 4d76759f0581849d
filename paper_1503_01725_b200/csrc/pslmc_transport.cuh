// pslmc_transport.cuh — k_photon and k_electron: persistent warps with lane refill, Woodcock photon
// flights with Klein–Nishina/Kahn Compton as a per-lane state machine, condensed-history electrons, the
// warp-staged electron queue, int64 fixed-point scoring.  PAPER.md:118-120 (iterated kernels), :161 (cut-offs);
// physics per DESIGN.md P1-P9.
#pragma once
#include "pslmc_kernels.cuh"

namespace pslmc {

// A queue of tracks: three 16-byte planes so every lane store/load is one 128-bit access.
struct Queue {
  float4 *a;            // x, y, z, E
  float4 *b;            // u, v, w, (unused)
  uint4  *c;            // hist_lo, hist_hi, track, (unused)
  unsigned *count;      // tail (device)
  unsigned cap;
};

enum { SRC_BUFFER = 0, SRC_QUEUE = 1 };
constexpr int kPhotonRefillMin = 8;            // k_photon likewise (r2: 1 -> 8 is 2-3 % of the kernel; 12, 16: slower)
constexpr int kElectronRefillMin = 8;          // k_electron refills in groups of >= 8 idle lanes (measured best of 1, 4, 8, 16)
constexpr unsigned kElectronChunk = 64;        // largest source chunk a k_electron warp reserves at once (r2: 32 -> 64 is 6 % of the kernel on C4: the cursor is one address for all warps)
constexpr int kXsIntervals = 4096;
constexpr size_t kAnnihBytes = 2 * sizeof(float4) * kThreads;   // k_photon: one pending annihilation photon per lane
constexpr size_t kXsBytes = sizeof(float) * (kXsHead + kXsIntervals + 4);     // head + n + 1 nodes, padded to 16 bytes

struct TransportArgs {
  Grid g;
  Control *ctl;
  unsigned long long seed;
  uint32_t ks[20];                    // Philox round keys of `seed` (host-computed)
  // source
  int src_kind;                       // SRC_BUFFER: p0/p1 planes from k_sample;  SRC_QUEUE: src queue
  int buffer_is_debug;                // SRC_BUFFER only: 1 = indexed by history, p1.w = status (skip < 0)
  const float4 *p0, *p1;
  const uint32_t *p2;                 // commissioning column per buffer entry, or null
  Queue src;
  const unsigned *src_count;          // entries available (device)
  unsigned *src_head;                 // consume cursor (device)
  unsigned long long first, n_total, perm_a;
  // sinks
  Queue eq;                           // sink of the charged secondaries
  // options
  unsigned long long *fp; unsigned long long fp_base;
  int electrons_local, static_lanes, stage_scoring;
  int fp_voxels;                      // DBG variants: strict fingerprints (MC_FLAG_FP_VOXELS)
  int want_type;                      // SRC_BUFFER, compact: take only entries of this particle type (bit 31 of p1.w)
  XsTable xs;                         // k_photon: cross-section table (global; copied to shared memory per CTA)
  const float *rhomax;                // largest density per material of this call's phantom (device; k_pack_phantom)
};

struct Tally {                         // per-thread running sums, flushed once at kernel exit
  unsigned long long inc, dep, esc;
  unsigned st[ST_COUNT];
};

template <bool DBG>
__device__ __forceinline__ void tally_flush(const TransportArgs &a, Tally &t) {
  unsigned long long inc = warp_sum_u64(t.inc), dep = warp_sum_u64(t.dep), esc = warp_sum_u64(t.esc);
  if ((threadIdx.x & 31) == 0) {
    unsigned long long (*L)[2] = a.ctl->ledger[(blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5)) % kLedgerSlots];
    add128(L[0], inc); add128(L[1], dep); add128(L[2], esc);
  }
  if (DBG) {
#pragma unroll
    for (int s = 0; s < ST_COUNT; ++s) {
      unsigned v = __reduce_add_sync(kFull, t.st[s]);
      if ((threadIdx.x & 31) == 0 && v) atomicAdd(&a.ctl->stat[s], (unsigned long long)v);
    }
  }
}

// Pending deposit: consecutive deposits into one voxel are merged before the atomic (integers: exact).
// Optional shared-memory staging of the scoring atomics (north_star (4), MC_FLAG_STAGE_SCORING): a per-CTA
// direct-mapped table of kScoreSlots voxel accumulators.  A voxel claims a free slot on first touch and keeps it
// for the whole launch (no eviction: integer sums make the result independent of who claimed what); deposits to
// a voxel that owns a slot are shared-memory atomics, all others go to the global grid as before; the table is
// added to the grid once at kernel exit.  Helps only where a launch concentrates its deposits on <~ 1e3 voxels
// per CTA (narrow beams); DESIGN.md §5 has the measured ablation.
constexpr int kScoreSlots = 1024;
constexpr size_t kScoreBytes = (size_t)kScoreSlots * (sizeof(unsigned long long) + sizeof(int));
template <bool ON>
struct ScoreStage {
  unsigned long long *sum; int *tag;                 // shared memory (unused when !ON)
  __device__ __forceinline__ void init(unsigned char *smem) {
    sum = nullptr; tag = nullptr;
    if (!ON) return;
    sum = reinterpret_cast<unsigned long long *>(smem); tag = reinterpret_cast<int *>(smem + sizeof(unsigned long long) * kScoreSlots);
    for (int i = threadIdx.x; i < kScoreSlots; i += kThreads) { sum[i] = 0ull; tag[i] = -1; }
    __syncthreads();
  }
  __device__ __forceinline__ void add(const Grid &g, int v, unsigned long long q) const {
    if (ON) {
      const unsigned s = ((unsigned)v * 2654435761u) >> 22;                       // 10 bits
      int t = tag[s];
      if (t == -1) { t = atomicCAS(tag + s, -1, v); if (t == -1) t = v; }
      if (t == v) { atomicAdd(sum + s, q); return; }
    }
    atomicAdd(g.acc + v, q);
  }
  __device__ __forceinline__ void drain(const Grid &g) const {                    // every thread of the CTA calls this
    if (!ON) return;
    __syncthreads();
    for (int i = threadIdx.x; i < kScoreSlots; i += kThreads)
      if (tag[i] >= 0 && sum[i]) atomicAdd(g.acc + tag[i], sum[i]);
  }
};

// Pending deposit: consecutive deposits into one voxel are merged before the atomic (integers: exact).
template <bool COM>                                   // COM: the kernel variants that may carry a commissioning tally (MODE_COM, MODE_DBG)
struct Pending {
  int v; long long q; uint32_t col;                  // col: commissioning column of the lane's current history
  template <bool ON> __device__ __forceinline__ void flush(const Grid &g, const ScoreStage<ON> &st) {
    if (q) {
      st.add(g, v, (unsigned long long)q);
      if (COM && g.com_index && ((__ldg(g.com_coarse + (v >> 14)) >> ((v >> 9) & 31)) & 1u) && ((__ldg(g.com_mask + (v >> 5)) >> (v & 31)) & 1u)) {
        const int row = __ldg(g.com_index + v);
        if (row > 0 && row <= g.com_rows) atomicAdd(g.com_dose + (size_t)col * g.com_rows + (row - 1), (unsigned long long)q);
      }
    }
    q = 0;
  }
  template <bool ON> __device__ __forceinline__ void add(const Grid &g, const ScoreStage<ON> &st, int vox, long long dq) {
    if (vox != v) { flush(g, st); v = vox; }
    q += dq;
  }
};

template <bool DBG>
__device__ __forceinline__ void finish_track(const TransportArgs &a, unsigned long long h, const Fnv &f) {
  if (DBG && a.fp) atomicAdd(a.fp + (h - a.fp_base), f.v);
}

// Warp-aggregated push through a per-warp shared-memory ring of 64 entries: lanes with `want` append at consecutive ring
// positions (ballot + prefix sum); whenever the ring holds >= 32 entries the warp writes 32 of them to the queue as three
// coalesced 512-byte rows.  Queue slots are taken 128 at a time with ONE tail atomic (four flushes per atomic: the tail is
// one address for every warp of the launch, and halving the atomics on it is worth more than the few null entries it
// costs); the part of a reservation a warp has not used when the kernel ends is filled with null entries (electrons of
// 1e-30 MeV, which k_electron ends in their first sub-step with a deposit of 0 quanta).  No atomic and no global store in
// the common iteration.  Convergent calls.
struct StageRing { float4 a[64], b[64]; uint4 c[64]; };           // 3 KiB per warp
struct StageCursor { unsigned head, n, base_raw, base, have; bool pending; };     // have: reserved slots not written yet (at `base`)
// The atomic's latency is not waited for: stage_reserve issues it (result left in lane 0's register), stage_resolve -
// one loop iteration later, or at kernel exit - broadcasts it.
__device__ __forceinline__ void stage_reserve(const Queue &q, StageCursor &sc, unsigned n_out) {
  if ((threadIdx.x & 31u) == 0) sc.base_raw = atomicAdd(q.count, n_out);
  sc.pending = true; sc.have = n_out;
}
__device__ __forceinline__ void stage_resolve(const Queue &q, Control *ctl, StageCursor &sc) {
  sc.base = __shfl_sync(kFull, sc.base_raw, 0);
  if (sc.base + sc.have > q.cap) { atomicOr(&ctl->overflow, 1u); sc.base = 0xffffffffu; }   // dropped whole; k_electron does not run on a queue that overflowed
  sc.pending = false;
}
// Writes the n_real oldest ring entries (and null entries up to n_out) to the next n_out reserved slots.
__device__ __forceinline__ void stage_write(const Queue &q, StageRing &r, StageCursor &sc, unsigned n_real, unsigned n_out) {
  const unsigned lane = threadIdx.x & 31u;
  __syncwarp();
  if (sc.base != 0xffffffffu && lane < n_out) {
    const unsigned p = (sc.head + lane) & 63u;
    const bool real = lane < n_real;
    // a null entry: an electron of 1e-30 MeV at a real entry's place - k_electron ends it in its first sub-step with a
    // deposit of 0 quanta (plain and commissioning variants only: with counters or fingerprints no half is left open)
    float4 A = r.a[real ? p : ((sc.head + sc.n - 1u) & 63u)]; if (!real) A.w = 1e-30f;
    __stcs(q.a + sc.base + lane, A);                                                        // write-once / read-once: streaming
    __stcs(q.b + sc.base + lane, real ? r.b[p] : make_float4(0.f, 0.f, 1.f, 0.f));
    __stcs(q.c + sc.base + lane, real ? r.c[p] : make_uint4(0u, 0u, 0u, 0u));
  }
  if (sc.base != 0xffffffffu) sc.base += n_out;
  sc.have -= n_out; sc.head = (sc.head + n_real) & 63u; sc.n -= n_real;
  __syncwarp();
}
// One call per loop iteration (convergent): resolves the reservation issued in the previous iteration, writes 32 entries
// when the ring holds that many and slots are at hand, appends this iteration's entries, and reserves 128 more slots once
// 32 entries are staged without any.  The ring never holds more than 31 + 32 entries.
__device__ __forceinline__ void stage_push(const Queue &q, Control *ctl, StageRing &r, StageCursor &sc, bool want,
                                           float4 A, float4 B, uint4 C, bool big) {
  if (sc.n >= 32u && sc.have) { if (sc.pending) stage_resolve(q, ctl, sc); stage_write(q, r, sc, 32u, 32u); }
  const unsigned m = __ballot_sync(kFull, want);
  if (m) {
    const unsigned lane = threadIdx.x & 31u;
    if (want) {
      const unsigned p = (sc.head + sc.n + __popc(m & ((1u << lane) - 1u))) & 63u;
      r.a[p] = A; r.b[p] = B; r.c[p] = C;
    }
    sc.n += __popc(m);
  }
  if (sc.n >= 32u && !sc.have) stage_reserve(q, sc, big ? 128u : 32u);      // (big: the warp still has source to come, so the second half will be used)
}
__device__ __forceinline__ void stage_drain(const Queue &q, Control *ctl, StageRing &r, StageCursor &sc) {
  if (sc.pending) stage_resolve(q, ctl, sc);
  while (sc.have) { const unsigned k = min(sc.n, 32u); stage_write(q, r, sc, k, 32u); }     // open halves: what is staged, then nulls
  if (sc.n) { const unsigned n = sc.n; stage_reserve(q, sc, n); stage_resolve(q, ctl, sc); stage_write(q, r, sc, n, n); }
}
// Refill protocol shared by both kernels: lanes without a track take the next source indices.  A warp
// takes `chunk` consecutive indices from the source cursor with ONE atomic and hands them out over
// the next refills (warp-uniform cursor in `sc`).  Returns the source index for this lane or
// 0xffffffff.  `exhausted` becomes true (warp-uniform) once the cursor passed the end.
struct SrcCursor { unsigned next, end, chunk; };          // chunk: size of the last reservation (shrinks towards the end of the source)
// Guided self-scheduling: the chunk shrinks with what was left at the warp's previous grab, so the
// last chunks are small and the warps finish together.
template <unsigned MAX_CHUNK>
__device__ __forceinline__ unsigned source_chunk(const TransportArgs &a, unsigned count, unsigned seen_end, unsigned need) {
  if (a.static_lanes) return 32u;
  const unsigned warps = gridDim.x * (kThreads / 32), left = count - min(count, seen_end);
  return min(MAX_CHUNK, max(need, (left / (warps * 2u)) & ~31u));     // near the end: exactly what the idle lanes need
}
// L2 prefetch of the source entries [first, end) a warp has just reserved (<= 128 entries = 16 lines per
// 16-byte plane): the loads of the following refills then find them on chip.
__device__ __forceinline__ void prefetch_chunk(const TransportArgs &a, unsigned n1, unsigned first, unsigned end) {
  const unsigned lane = threadIdx.x & 31u, e = first + (lane & 15u) * 8u;       // 8 entries per 128-byte line
  if (e >= end) return;
  const void *p0, *p1, *p2 = nullptr;
  if (a.src_kind == SRC_BUFFER && e < n1) { p0 = a.p0 + e; p1 = a.p1 + e; }
  else { const unsigned q = a.src_kind == SRC_BUFFER ? e - n1 : e; p0 = a.src.a + q; p1 = a.src.b + q; p2 = a.src.c + q; }
  asm volatile("prefetch.global.L2 [%0];" ::"l"(lane < 16u ? p0 : p1));
  if (p2 && lane < 16u) asm volatile("prefetch.global.L2 [%0];" ::"l"(p2));
}
template <int MIN_IDLE, unsigned MAX_CHUNK>
__device__ __forceinline__ unsigned refill_index(const TransportArgs &a, bool idle, unsigned n1, unsigned count, SrcCursor &sc, bool &exhausted) {
  const unsigned need = __ballot_sync(kFull, idle);
  if (!need || exhausted) return 0xffffffffu;
  if (MIN_IDLE > 1 && need != kFull && __popc(need) < MIN_IDLE) return 0xffffffffu;   // refill in groups: the refill code then runs with more lanes
  if (a.static_lanes && need != kFull) return 0xffffffffu;       // ablation: a warp refills only when all lanes are done
  const unsigned lane = threadIdx.x & 31u;
  if (sc.next >= sc.end) {
    const unsigned chunk = source_chunk<MAX_CHUNK>(a, count, sc.end, __popc(need));
    unsigned base = 0;
    if (lane == 0) base = atomicAdd(a.src_head, chunk);
    base = __shfl_sync(kFull, base, 0);
    if (base >= count) { exhausted = true; return 0xffffffffu; }
    sc.next = base; sc.end = min(base + chunk, count); sc.chunk = chunk;
    prefetch_chunk(a, n1, sc.next, sc.end);
  }
  const unsigned rank = __popc(need & ((1u << lane) - 1u)), avail = sc.end - sc.next;
  const unsigned idx = sc.next + rank;
  sc.next += min((unsigned)__popc(need), avail);
  return (idle && rank < avail) ? idx : 0xffffffffu;
}

struct TrackIn { float x, y, z, u, v, w, E; unsigned long long h; uint32_t track, blk, col; bool ok; };

__device__ __forceinline__ TrackIn load_track(const TransportArgs &a, unsigned idx, unsigned n1) {
  TrackIn t;
  if (a.src_kind == SRC_BUFFER) {
    const float4 A = __ldcs(a.p0 + idx), B = __ldcs(a.p1 + idx);
    t.x = A.x; t.y = A.y; t.z = A.z; t.E = A.w; t.u = B.x; t.v = B.y; t.w = B.z;
    unsigned long long tt;
    if (a.buffer_is_debug) {
      tt = idx; t.ok = B.w >= 0.0f;
      if (t.ok && !(A.w >= 0.0f && A.w < 4096.0f)) { t.ok = false; a.ctl->bad_input = 1u; }     // warp_sum_q is exact below 4096 MeV
    }
    else { const unsigned bits = __float_as_uint(B.w); tt = bits & 0x7fffffffu; t.ok = (int)(bits >> 31) == a.want_type; }
    t.h = history_of(a.first + tt, a.perm_a, a.n_total);
    t.track = 0u; t.blk = 2u; t.col = a.p2 ? a.p2[idx] : 0u;      // blocks 0, 1 were the source draws
  } else {
    const float4 A = __ldcs(a.src.a + idx), B = __ldcs(a.src.b + idx); const uint4 C = __ldcs(a.src.c + idx);
    t.x = A.x; t.y = A.y; t.z = A.z; t.E = A.w; t.u = B.x; t.v = B.y; t.w = B.z;
    t.h = ((unsigned long long)C.y << 32) | C.x; t.track = C.z; t.blk = 0u; t.col = C.w; t.ok = true;
  }
  return t;
}


// ------------------------------------------------------------------ k_photon
// One lane = one photon track at a time, as a small state machine.  Every loop iteration runs at most
// two "events" per lane, each with ONE Philox generation site shared by all lanes of the warp:
//   event 1 (state FLIGHT): cut-off test, Woodcock flight (draws a, b), voxel fetch, interaction choice;
//   event 2 (state KAHN / PAIR): one Kahn trial (3 draws, + the azimuth draw when it is accepted, then the
//            Compton kinematics) or the pair-production split (3 draws).
// A lane whose Kahn trial is rejected retries in the next iteration while its neighbours fly, instead
// of holding the warp in a rejection loop.  Cross-sections come from the shared-memory table.
enum { PH_IDLE = 0, PH_FLIGHT = 1, PH_KAHN = 2, PH_PAIR = 3 };

// MODE: kernel variant - MODE_PLAIN (what bench.py times), MODE_COM (plain + the commissioning tally: every track carries
// the PSR column of its history), MODE_DBG (event counters, fingerprints, and the tally when asked for).
enum { MODE_PLAIN = 0, MODE_COM = 1, MODE_DBG = 2 };
template <int MODE, bool STAGE>
__global__ void __launch_bounds__(kThreads, 3) k_photon(const __grid_constant__ TransportArgs a) {
  constexpr bool DBG = MODE == MODE_DBG, COM = MODE != MODE_PLAIN;
  extern __shared__ __align__(16) unsigned char s_raw[];           // [xs table | one StageRing per warp]
  float *s_xs = reinterpret_cast<float *>(s_raw);
  for (int i = threadIdx.x; i <= a.xs.n; i += kThreads) s_xs[kXsHead + i] = a.xs.data[kXsHead + i];
  if (threadIdx.x < 3) {                                 // Woodcock majorant coefficients of this phantom (k_pack_phantom's rhomax)
    const float rm = a.rhomax[threadIdx.x];
    s_xs[4 * threadIdx.x] = rm * c_mat.ne[threadIdx.x]; s_xs[4 * threadIdx.x + 1] = rm * c_mat.cphoto[threadIdx.x];
    s_xs[4 * threadIdx.x + 2] = rm * c_mat.ppair[threadIdx.x]; s_xs[4 * threadIdx.x + 3] = 0.0f;
  }
  __syncthreads();
  // the second annihilation photon of a pair waits here, one slot per lane: (x, y, z, track id), (u, v, w, -)
  float4 *s_annih = reinterpret_cast<float4 *>(s_raw + kXsBytes + sizeof(StageRing) * (kThreads / 32)) + 2 * threadIdx.x;
  ScoreStage<STAGE> stage; stage.init(s_raw + kXsBytes + sizeof(StageRing) * (kThreads / 32) + kAnnihBytes);
  const Grid &g = a.g;
  const bool bricks = use_bricks(g);
  const unsigned n1 = a.src_kind == SRC_QUEUE ? min(*a.src_count, a.src.cap) : *a.src_count;
  const unsigned count = n1;
  SrcCursor sc; sc.next = sc.end = sc.chunk = 0u;
  StageRing &ring = *reinterpret_cast<StageRing *>(s_raw + kXsBytes + sizeof(StageRing) * (threadIdx.x >> 5));
  StageCursor stg; stg.head = stg.n = stg.base_raw = stg.base = stg.have = 0u; stg.pending = false;
  Tally tl; tl.inc = tl.dep = tl.esc = 0;
  if (DBG) { for (int s = 0; s < ST_COUNT; ++s) tl.st[s] = 0; }
  Pending<COM> pend; pend.v = 0; pend.q = 0; pend.col = 0u;
  int state = PH_IDLE; bool exhausted = false, collided = false, pend2 = false;
  float x = 0, y = 0, z = 0, u = 0, v = 0, w = 1, E = 0;
  int cvox = 0;                                          // voxel of the current position
  unsigned long long h = 0; uint32_t nchild = 0;
  Rng rng; rng.init(0ull, 0u, 0u);
  Fnv fnv; fnv.v = 0;

  for (;;) {
    // ---- a lane whose photon ended and that still holds the second annihilation photon of a pair takes that one
    if (state == PH_IDLE && pend2) {
      const float4 A = s_annih[0], Bv = s_annih[1];
      x = A.x; y = A.y; z = A.z; u = Bv.x; v = Bv.y; w = Bv.z; E = kEAnnih; nchild = 0; collided = false; pend2 = false;
      rng.init(h, __float_as_uint(A.w), 0u);
      if (DBG) fnv.init(__float_as_uint(A.w));
      int vi, vj, vk; locate(g, x, y, z, vi, vj, vk);       // the conversion site: inside the grid
      cvox = vox_index(g, vi, vj, vk); state = PH_FLIGHT;
    }
    // ---- refill idle lanes
    const unsigned idx = refill_index<kPhotonRefillMin, 128u>(a, state == PH_IDLE, n1, count, sc, exhausted);
    if (idx != 0xffffffffu) {
      const TrackIn t = load_track(a, idx, n1);
      if (t.ok) {
        x = t.x; y = t.y; z = t.z; u = t.u; v = t.v; w = t.w; E = t.E; h = t.h; nchild = 0; collided = false;
        if (COM && g.com_index) { pend.flush(g, stage); pend.col = t.col; }
        rng.init(h, t.track, t.blk);
        if (DBG) fnv.init(t.track);
        if (a.buffer_is_debug) tl.inc += (unsigned long long)quanta(E);
        int vi, vj, vk;
        // only the debug buffer holds tracks outside the grid: k_sample already moved the primaries to
        // their entry points, and queued secondaries are born inside
        bool in = locate(g, x, y, z, vi, vj, vk);
        if (!in && a.buffer_is_debug) in = enter(g, x, y, z, u, v, w, vi, vj, vk);
        if (!in) {
          tl.esc += (unsigned long long)quanta(E);
          if (DBG) { fnv.byte('M'); ++tl.st[ST_MISSED]; finish_track<DBG>(a, h, fnv); }
        } else { cvox = vox_index(g, vi, vj, vk); state = PH_FLIGHT; }
      }
    }
    if (!__any_sync(kFull, state != PH_IDLE)) { if (exhausted) break; else continue; }

    // ---- event 1: one Woodcock flight and the choice of interaction
    if (state == PH_FLIGHT) {
      bool done = false;
      float skn = 0.f, inv_e3 = 0.f, lp2 = 0.f, mu_max = 0.f;
      if (E >= kPcut) xs_lookup(s_xs, a.xs.x0, a.xs.inv_h, a.xs.n, E, skn, inv_e3, lp2, mu_max);
      if (E < kPcut) {                                   // below cut-off: absorbed on the spot
        const long long q = quanta(E); pend.add(g, stage, cvox, q); tl.dep += (unsigned long long)q;
        if (DBG) { if (a.fp_voxels) fnv.u32((uint32_t)cvox); fnv.byte('A'); ++tl.st[ST_PCUT]; ++tl.st[ST_DEPOSITS]; }
        done = true;
      } else if (!(mu_max > 0.0f)) {
        tl.esc += (unsigned long long)quanta(E);
        if (DBG) { fnv.byte('E'); ++tl.st[ST_PESC]; if (!collided && rng.track == 0u) ++tl.st[ST_UNCOLLIDED]; }
        done = true;
      } else {
        uint32_t d0, d1, d2, d3;
        rng.next(a.ks, d0, d1, d2, d3);                  // flight block: free path, choice of interaction
        const float s = -logf(u_oc(d0)) / mu_max;
        x = __fmaf_rn(s, u, x); y = __fmaf_rn(s, v, y); z = __fmaf_rn(s, w, z);
        if (DBG) ++tl.st[ST_FLIGHTS];
        int vi, vj, vk;
        if (!locate(g, x, y, z, vi, vj, vk)) {
          tl.esc += (unsigned long long)quanta(E);
          if (DBG) { fnv.byte('E'); ++tl.st[ST_PESC]; if (!collided && rng.track == 0u) ++tl.st[ST_UNCOLLIDED]; }
          done = true;
        } else {
          cvox = vox_index(g, vi, vj, vk);
          float rho; int mt; fetch_voxel(g, bricks, vi, vj, vk, cvox, rho, mt);
          const float muC = rho * (c_mat.ne[mt] * skn), muT = rho * (c_mat.cphoto[mt] * inv_e3), muK = rho * (c_mat.ppair[mt] * lp2);
          const float tt = u_co(d1) * mu_max;
          if (tt < muC) {                                // Compton: Kahn trials are event 2
            collided = true; state = PH_KAHN;
            if (DBG) { fnv.byte('C'); ++tl.st[ST_COMPTON]; }
          } else if (tt < muC + muT) {                   // photo-electric: local absorption
            const long long q = quanta(E); pend.add(g, stage, cvox, q); tl.dep += (unsigned long long)q;
            if (DBG) { fnv.byte('P'); if (a.fp_voxels) fnv.u32((uint32_t)cvox); ++tl.st[ST_PHOTO]; ++tl.st[ST_DEPOSITS]; }
            done = true;
          } else if (tt < muC + muT + muK) {             // pair production: event 2
            state = PH_PAIR;
            if (DBG) { fnv.byte('X'); ++tl.st[ST_PAIR]; }
          } else if (DBG) { fnv.byte('V'); ++tl.st[ST_VIRTUAL]; }
        }
      }
      if (done) { if (DBG) finish_track<DBG>(a, h, fnv); state = PH_IDLE; }
    }

    // ---- event 2: one Kahn trial (+ Compton kinematics when accepted) or the pair split
    bool push_e = false, push_p = false; float ex = 0, ey = 0, ez = 0, eT = 0; uint32_t etrack = 0;
    float pairT[2] = {0.f, 0.f};
    if (state >= PH_KAHN) {
      uint32_t d0, d1, d2, d3;
      rng.gen(a.ks, rng.blk, d0, d1, d2, d3);            // trial block (r1, r2, r3, azimuth) or pair block (split, cos, azimuth)
      if (state == PH_KAHN) {
        // Kahn's rejection (P5), TWO trials per event: the blocks of this and of the next trial are generated
        // side by side (independent instruction streams), the first accepted one is used and the stream advances past it;
        // a track needs 1.2 events per scatter instead of 1.7 and the flight section of the next iteration runs fuller.
        // With dn = 1 + 2 alpha r2:  branch A: eta = dn, branch B: eta = (2 alpha + 1)/dn.  k = (eta - 1)/alpha is
        // 2 r2 (A) or 2 (1 - r2)/dn (B) in exact arithmetic; these forms have no cancellation in fp32.
        uint32_t e0, e1, e2, e3;
        rng.gen(a.ks, rng.blk + 1u, e0, e1, e2, e3);
        const float ta = E * (2.0f / kMe), tp1 = ta + 1.0f, thr = __fdividef(tp1, ta + 9.0f);      // 2 alpha
        bool brA, accept; float ie, k, ct;
        auto trial = [&](uint32_t w0, uint32_t w1, uint32_t w2, bool &bA, float &ie_, float &k_, float &ct_) {
          const float r1 = u_co(w0), r2 = u_co(w1), r3 = u_co(w2);
          const float dn = __fmaf_rn(ta, r2, 1.0f), idn = rcp_fast(dn);
          bA = r1 <= thr;
          ie_ = bA ? idn : __fdividef(dn, tp1);                          // 1/eta
          k_ = bA ? 2.0f * r2 : 2.0f * (1.0f - r2) * idn;                // 1 - cos(theta)
          ct_ = 1.0f - k_;
          return bA ? (r3 <= 4.0f * (ie_ - ie_ * ie_)) : (r3 <= 0.5f * (ct_ * ct_ + ie_));
        };
        bool brA2; float ie2, k2, ct2;
        const bool acc1 = trial(d0, d1, d2, brA, ie, k, ct), acc2 = trial(e0, e1, e2, brA2, ie2, k2, ct2) && !acc1;
        if (acc2) { brA = brA2; ie = ie2; k = k2; ct = ct2; d3 = e3; }
        accept = acc1 || acc2;
        rng.blk += acc1 ? 1u : 2u;
        if (DBG) tl.st[ST_KAHN] += acc1 ? 1u : 2u;
        if (accept) {
          if (DBG && a.fp_voxels) fnv.u32(rng.blk | (brA ? 0u : 0x80000000u));     // strict fingerprint: which trial was accepted, on which branch
          const float sn = sqrt_fast(fmaxf(0.0f, k * (2.0f - k)));
          const float Ep = E * ie, T = E - Ep, u0 = u, v0 = v, w0 = w;
          rotate(u, v, w, ct, sn, u_co(d3));
          if (T >= kEcut && !a.electrons_local) {
            const float dxe = E * u0 - Ep * u, dye = E * v0 - Ep * v, dze = E * w0 - Ep * w;
            const float n2 = dxe * dxe + dye * dye + dze * dze;
            if (n2 > 0.0f) { const float inv = rsqrtf(n2); ex = dxe * inv; ey = dye * inv; ez = dze * inv; }
            else { ex = u0; ey = v0; ez = w0; }
            eT = T; etrack = child_track(rng.track, nchild, 0u); push_e = true;
            if (DBG) ++tl.st[ST_SEC_E];
          } else {
            const long long q = quanta(T); pend.add(g, stage, cvox, q); tl.dep += (unsigned long long)q;
            if (DBG) { if (a.fp_voxels) fnv.u32((uint32_t)cvox); ++tl.st[ST_DEPOSITS]; }
          }
          ++nchild; E = Ep; state = PH_FLIGHT;
        }
      } else {                                           // pair production: the pushes happen below, convergently
        ++rng.blk;
        const float Tsum = E - kEPair, Tm = u_co(d0) * Tsum, Tp = Tsum - Tm;
        const float Tc[2] = {Tm, Tp};
#pragma unroll
        for (int sl = 0; sl < 2; ++sl) {
          if (Tc[sl] >= kEcut && !a.electrons_local) {
            pairT[sl] = Tc[sl];
            if (DBG) ++tl.st[ST_SEC_E];
          } else {
            const long long q = quanta(Tc[sl]); pend.add(g, stage, cvox, q); tl.dep += (unsigned long long)q;
            if (DBG) { if (a.fp_voxels) fnv.u32((uint32_t)cvox); ++tl.st[ST_DEPOSITS]; }
          }
        }
        const float cz = 2.0f * u_co(d1) - 1.0f, sz = sqrtf(fmaxf(0.0f, 1.0f - cz * cz));
        float sa, ca; sincospif(2.0f * u_co(d2), &sa, &ca);
        ex = sz * ca; ey = sz * sa; ez = cz; push_p = true;
        if (DBG) { tl.st[ST_SEC_P] += 2; finish_track<DBG>(a, h, fnv); }
        state = PH_IDLE;
      }
    }
    // ---- secondaries, convergent: Compton electrons through the staging ring ...
    const bool big = !DBG && !exhausted && sc.chunk >= 128u;   // not in the tail of the source: queue slots are taken 128 at a time
    stage_push(a.eq, a.ctl, ring, stg, push_e, make_float4(x, y, z, eT), make_float4(ex, ey, ez, 0.f),
               make_uint4((uint32_t)h, (uint32_t)(h >> 32), etrack, COM ? pend.col : 0u), big);
    // ... and, in the rare iteration with a pair production in the warp, the e-/e+ through the same ring (the lane's
    // x, y, z, u, v, w, h, track and nchild are still those of the converting photon)
    const unsigned mp = __ballot_sync(kFull, push_p);
    if (mp) {
#pragma unroll
      for (int sl = 0; sl < 2; ++sl)
        stage_push(a.eq, a.ctl, ring, stg, pairT[sl] > 0.0f, make_float4(x, y, z, pairT[sl]), make_float4(u, v, w, 0.f),
                   make_uint4((uint32_t)h, (uint32_t)(h >> 32), child_track(rng.track, nchild, (uint32_t)sl), COM ? pend.col : 0u), big);
      // the two 0.511 MeV annihilation photons (tracks: slots 2, 3 of this conversion) stay in the lane: it continues
      // as the first at once and keeps the second in its shared-memory slot until the first has ended
      if (push_p) {
        const uint32_t t1 = child_track(rng.track, nchild, 2u), t2 = child_track(rng.track, nchild, 3u);
        s_annih[0] = make_float4(x, y, z, __uint_as_float(t2)); s_annih[1] = make_float4(-ex, -ey, -ez, 0.f);
        pend2 = true;
        u = ex; v = ey; w = ez; E = kEAnnih; nchild = 0; collided = false;
        rng.init(h, t1, 0u);
        if (DBG) fnv.init(t1);
        state = PH_FLIGHT;
      }
    }
  }
  stage_drain(a.eq, a.ctl, ring, stg);
  pend.flush(g, stage);
  stage.drain(g);
  tally_flush<DBG>(a, tl);
}

// ------------------------------------------------------------------ k_electron
// Electrons carry (voxel index, offset inside the voxel) instead of global coordinates: fp32 then
// resolves positions to ~3e-8 cm relative to the voxel faces that decide every step, instead of the
// ~1e-6 cm of a global coordinate.  In exact arithmetic this is the
// same walk as floor((pos - o)/d) on global coordinates.  One loop iteration = one sub-step; the two
// draws of a condensed step come from one Philox site (draw numbers are always even here).
template <int MODE, bool STAGE>
__global__ void __launch_bounds__(kThreads, 4) k_electron(const __grid_constant__ TransportArgs a) {
  constexpr bool DBG = MODE == MODE_DBG, COM = MODE != MODE_PLAIN;
  extern __shared__ __align__(16) unsigned char s_raw[];           // [score staging table] when enabled
  const Grid &g = a.g;
  // a queue that overflowed holds slots that were never written (a reservation that straddled its end is dropped
  // whole): the call fails with MC_E_OVERFLOW, nothing here may be read
  if (a.src_kind == SRC_QUEUE && (a.ctl->overflow & 1u)) return;
  ScoreStage<STAGE> stage; stage.init(s_raw);
  const bool bricks = use_bricks(g);
  const unsigned n1 = a.src_kind == SRC_QUEUE ? min(*a.src_count, a.src.cap) : *a.src_count;
  const unsigned count = n1;
  SrcCursor sc; sc.next = sc.end = sc.chunk = 0u;
  Tally tl; tl.inc = tl.dep = tl.esc = 0;
  if (DBG) { for (int s = 0; s < ST_COUNT; ++s) tl.st[s] = 0; }
  Pending<COM> pend; pend.v = 0; pend.q = 0; pend.col = 0u;
  bool active = false, exhausted = false;
  float lx = 0, ly = 0, lz = 0, u = 0, v = 0, w = 1, T = 0;      // offset inside voxel (vi,vj,vk), direction, energy
  float iu = 0, iv = 0, iw = 1;                                   // reciprocal direction cosines (refreshed when the direction changes)
  int vi = 0, vj = 0, vk = 0;
  unsigned long long h = 0; uint32_t steps = 0;
  // condensed step (P7): energy still to lose in it, rho*s/X0 accumulated, energy at its start
  float budget = 0, tacc = 0, Tms = 0; bool fresh = true;
  Rng rng; rng.init(0ull, 0u, 0u);
  Fnv fnv; fnv.v = 0;

  for (;;) {
    const unsigned idx = refill_index<kElectronRefillMin, kElectronChunk>(a, !active, n1, count, sc, exhausted);
    if (idx != 0xffffffffu) {
      const TrackIn t = load_track(a, idx, n1);
      if (t.ok) {
        float x = t.x, y = t.y, z = t.z;
        u = t.u; v = t.v; w = t.w; T = t.E; h = t.h; steps = 0; fresh = true;
        if (COM && g.com_index) { pend.flush(g, stage); pend.col = t.col; }
        rng.init(h, t.track, t.blk);
        if (DBG) { fnv.init(t.track); ++tl.st[ST_ETRACKS]; }
        if (a.buffer_is_debug) tl.inc += (unsigned long long)quanta(T);
        active = true;
        bool in = locate(g, x, y, z, vi, vj, vk);
        if (!in && a.buffer_is_debug) in = enter(g, x, y, z, u, v, w, vi, vj, vk);
        if (!in) {
          tl.esc += (unsigned long long)quanta(T);
          if (DBG) { fnv.u32(0u); fnv.byte('M'); ++tl.st[ST_MISSED]; finish_track<DBG>(a, h, fnv); }
          active = false;
        } else {
          lx = (x - g.ox) - (float)vi * g.dx; ly = (y - g.oy) - (float)vj * g.dy; lz = (z - g.oz) - (float)vk * g.dz;
          iu = rcp_fast(u); iv = rcp_fast(v); iw = rcp_fast(w);
        }
      }
    }
    if (!__any_sync(kFull, active)) { if (exhausted) break; else continue; }

    if (active) {                                        // one sub-step
      const int vox = vox_index(g, vi, vj, vk);
      float rho; int mt; fetch_voxel(g, bricks, vi, vj, vk, vox, rho, mt);
      if (fresh) { budget = kFe * T; Tms = T; tacc = 0.0f; fresh = false; }
      const float D = (c_mat.sscale[mt] * rho) * __fmaf_rn(0.078f, T, __fmaf_rn(0.25f, rcp_fast(T), 1.52f));
      const float sE = D > 0.0f ? __fdividef(budget, D) : INFINITY;
      // distance to the exit face of this voxel (a zero direction component never limits)
      const float sx = (u > 0.0f ? g.dx - lx : -lx) * iu, sy = (v > 0.0f ? g.dy - ly : -ly) * iv, sz = (w > 0.0f ? g.dz - lz : -lz) * iw;
      float sv = fminf(fminf(u != 0.0f ? sx : INFINITY, v != 0.0f ? sy : INFINITY), w != 0.0f ? sz : INFINITY);
      sv = fmaxf(sv, 0.0f);
      const bool turn = sE <= sv + kEpsB;              // this sub-step ends the condensed step
      const float s = turn ? sE : sv + kEpsB, dT = turn ? budget : D * s;
      ++steps;
      if (DBG) { ++tl.st[ST_ESTEPS]; ++tl.st[ST_DEPOSITS]; if (a.fp_voxels) fnv.u32((uint32_t)vox | (turn ? 0x80000000u : 0u)); }
      bool done = false;
      const bool stop = T - dT <= kEcut;               // below the cut-off after this sub-step: everything left is deposited here
      const long long q = quanta(stop ? T : dT); pend.add(g, stage, vox, q); tl.dep += (unsigned long long)q;
      if (stop) {
        if (DBG) { fnv.u32(steps); fnv.byte('A'); }
        done = true;
      } else {
        lx = __fmaf_rn(s, u, lx); ly = __fmaf_rn(s, v, ly); lz = __fmaf_rn(s, w, lz);
        T -= dT; budget -= dT; tacc = __fmaf_rn(rho * s, c_mat.inv_x0[mt], tacc);
        // re-home: a step ends at most eps beyond the face it was limited by
        if (lx >= g.dx) { lx -= g.dx; ++vi; } else if (lx < 0.0f) { lx += g.dx; --vi; }
        if (ly >= g.dy) { ly -= g.dy; ++vj; } else if (ly < 0.0f) { ly += g.dy; --vj; }
        if (lz >= g.dz) { lz -= g.dz; ++vk; } else if (lz < 0.0f) { lz += g.dz; --vk; }
        if ((unsigned)vi >= (unsigned)g.nx || (unsigned)vj >= (unsigned)g.ny || (unsigned)vk >= (unsigned)g.nz) {
          tl.esc += (unsigned long long)quanta(T);
          if (DBG) { fnv.u32(steps); fnv.byte('E'); ++tl.st[ST_EESC]; }
          done = true;
        } else if (turn) {
          uint32_t d0, d1, d2, d3;
          rng.next(a.ks, d0, d1, d2, d3);                // deflection block: Gaussian radius, azimuth
          if (DBG) ++tl.st[ST_DEFLECT];
          // theta = (13.6 / p beta) sqrt(tacc) sqrt(-2 ln a), p beta = Tms (Tms + 2 me)/(Tms + me): one division, one root
          const float c = __fdividef(13.6f * (Tms + kMe), Tms * (Tms + 2.0f * kMe));
          const float th = fminf(kPi, c * sqrt_fast(tacc * (-2.0f * __logf(u_oc(d0)))));
          float st, ct; __sincosf(th, &st, &ct);               // th in [0, pi]: SFU path, abs error ~4e-7
          rotate(u, v, w, ct, st, u_co(d1));
          iu = rcp_fast(u); iv = rcp_fast(v); iw = rcp_fast(w);
          fresh = true;
        }
      }
      if (done) { if (DBG) finish_track<DBG>(a, h, fnv); active = false; }
    }
  }
  pend.flush(g, stage);
  stage.drain(g);
  tally_flush<DBG>(a, tl);
}

}  // namespace pslmc
