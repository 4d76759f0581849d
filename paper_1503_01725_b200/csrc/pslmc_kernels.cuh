// pslmc_kernels.cuh — k_sample (PAPER.md:82-116 S3-S5: alias pick, position, energy, direction, jaw test, set-up
// transform, phantom entry, compaction of the survivors), the control block, phantom packing, finalise.
#pragma once
#include "pslmc_device.cuh"

namespace pslmc {

constexpr int kThreads = 256;
constexpr int kLedgerSlots = 32;
constexpr unsigned kFull = 0xffffffffu;

enum Stat {
  ST_MISSED = 0, ST_FLIGHTS, ST_VIRTUAL, ST_COMPTON, ST_PHOTO, ST_PAIR, ST_PCUT, ST_PESC, ST_UNCOLLIDED,
  ST_SEC_E, ST_SEC_P, ST_ETRACKS, ST_ESTEPS, ST_EESC, ST_DEPOSITS, ST_KAHN, ST_DEFLECT, ST_COUNT
};

// Device-resident control block.  `batch` part is reset by k_next_batch, the rest once per call.
struct Control {
  // per batch
  unsigned n_pb, head_pb;          // particle buffer: entries written by k_sample, consume cursor
  unsigned n_eq, head_eq;          // electron queue
  unsigned head_pb_e;              // mixed order: consume cursor of the electron pass over the particle buffer
  // per call
  unsigned overflow;               // bit 0: the electron queue was full; bit 1: a voxel accumulator wrapped → MC_E_OVERFLOW
  unsigned bad_input;              // mc_transport_debug: a particle with an energy outside [0, 4096) MeV was skipped
  unsigned hw_eq;                  // electron-queue high-water mark
  unsigned long long n_accepted;   // primaries that passed the jaws and entered the phantom
  unsigned long long n_missed;     // primaries that passed the jaws but missed the phantom (k_sample, compact mode)
  unsigned long long ledger[kLedgerSlots][4][2];   // [slot][incident,deposited,escaped,jaw][lo,hi] quanta
  unsigned long long stat[ST_COUNT];
  float rhomax[4];                 // largest density per material (as float, written via atomicMax on bits)
  unsigned n_uniform_bricks;       // bricks of 4x4x4 voxels whose voxels are all equal (k_bricks; hierarchical phantom)
  unsigned n_uniform_sbricks;      // super-bricks of 4x4x4 bricks that are one uniform region (k_sbricks)
};

// One alias-table entry, 16 B: everything k_sample needs after picking a column.
struct __align__(16) AliasEntry {
  uint32_t thresh;                 // accept column if frac < thresh
  uint16_t ring_c, sector_c;       // the column's own let
  uint16_t ring_a, sector_a;       // the alias let
  uint32_t pad;
};

struct SourceModel {               // read-only, uploaded once by psl_build
  const AliasEntry *table;         // all groups back to back
  const uint32_t *let_off;         // [G] first entry of group g
  const uint32_t *n_let;           // [G]
  int n_groups, n_ebin, n_sectors;
  int let_mode;                    // 0: ring sectors; 1: Cartesian grid of square lets (entries hold Xbin, Ybin)
  float grid_x0, let_size;
  float e_min, e_bin_width, ring_width, z_phsp, inv_nsec;
  float sigma_src[3], z_src[3];
  int particle_type[3];
  float jaw_tx[3], jaw_ty[3];      // (z_jx - z_s)/(z_p - z_s), (z_jy - z_s)/(z_p - z_s)
  float jx_lo, jx_hi, jy_lo, jy_hi;   // jaw edges on their own planes
  // Eq. 6 / Eq. 7 direction models, K = 0: focal geometry.  {P_cum, mu, sigma_a, sigma_b}[ebin][ring][K]
  const float4 *dir_tab[3];
  int dir_K[3], n_ring;
  float jaw_dzx, jaw_dzy;             // z_jx - z_p, z_jy - z_p
};

struct BeamXf { float iso[3]; float R[9]; float sad; };
struct TileMap { int shift, ntx, nty, nbins; };      // entry tiles (below); nbins = 0: no ordering

struct SampleArgs {
  SourceModel m;
  BeamXf beam;
  unsigned long long off_g[160];     // [G+1] prefix offsets of the groups' history-id ranges (Eq. 3; host-computed, G <= 159)
  uint32_t ks[20];                   // Philox round keys of `seed` (host-computed)
  unsigned long long seed, first, n_total, perm_a;   // perm_a != 0 → mixed order: h = (perm_a * t) mod n_total
  unsigned count;
  float4 *p0, *p1;                   // outputs (two float4 planes)
  uint32_t *p2;                      // compact mode, commissioning tally: column (PSR unit) of every packed particle, or null
  Control *ctl;
  unsigned long long *fp;            // fingerprints or null
  unsigned long long fp_base;
  int compact;                       // 1: survivors packed, p1.w = local index bits; 0: indexed by t, p1.w = status
  Grid g;                            // compact mode: survivors are moved to their phantom entry point here (P4),
  int stats;                         //   with every lane of the warp busy, instead of in the transport kernels' refill
  TileMap tm; unsigned *tile_count;  // compact mode, tile ordering: entry-tile histogram of the batch (device), or null
};

__device__ __forceinline__ unsigned long long history_of(unsigned long long t, unsigned long long perm_a, unsigned long long n_total) {
  return perm_a ? (perm_a * t) % n_total : t;
}

// ------------------------------------------------------------------ entry tiles (the spatial inner loop)
// A batch's survivors can be ordered by the tile of the phantom their entry voxel lies in, so that the lanes resident at
// any time work under a few neighbouring tiles and their voxel gathers and scoring atomics stay in L2.
// Tiles are cubes of 2^shift voxels; bins run in snake order (x reversed on odd rows, y reversed on odd slabs) so that
// consecutive bins are always face neighbours.  Counting sort: k_sample counts, k_tile_scan turns counts into
// cursors, k_tile_scatter moves the particles.  The order inside a bin is arbitrary: results do not depend on it.
constexpr int kTileBinsMax = 4096;
__device__ __forceinline__ unsigned tile_bin(const TileMap &tm, int vi, int vj, int vk) {
  int tx = vi >> tm.shift, ty = vj >> tm.shift; const int tz = vk >> tm.shift;
  if (tz & 1) ty = tm.nty - 1 - ty;
  const int row = ty + tm.nty * tz;
  if (row & 1) tx = tm.ntx - 1 - tx;
  return (unsigned)(tx + tm.ntx * row);
}

// ------------------------------------------------------------------ k_sample
// Persistent grid: a thread samples histories t = blockIdx.x*2*kThreads + {0, kThreads} + threadIdx.x + i*gridDim.x*2*kThreads.  The
// (sub-source, energy bin) group of a history is found once per thread and then walked forward (sorted order:
// history ids only grow), ledgers are summed in registers and flushed once per warp at the end: no barrier in the loop.
__global__ void __launch_bounds__(kThreads) k_sample(const __grid_constant__ SampleArgs a) {
  __shared__ unsigned long long s_off[160];
  extern __shared__ unsigned s_hist[];                     // [tm.nbins] entry-tile histogram of this CTA (tile ordering only)
  const SourceModel &m = a.m;
  for (int i = threadIdx.x; i <= m.n_groups; i += kThreads) s_off[i] = a.off_g[i];      // (constant bank → shared: indexed divergently below)
  const bool tiles = a.tm.nbins > 0 && a.tile_count != nullptr;
  if (tiles) for (int i = threadIdx.x; i < a.tm.nbins; i += kThreads) s_hist[i] = 0u;
  __syncthreads();
  const unsigned lane = threadIdx.x & 31u;
  unsigned long long q_inc = 0, q_jaw = 0, q_esc = 0;
  unsigned n_miss = 0;
  int g = -1;                                              // group of the thread's previous history (sorted order)
  // two histories per thread and iteration (t and t + kThreads): one buffer-tail atomic per 64 histories of a warp
  for (unsigned t0 = blockIdx.x * (2 * kThreads); t0 < a.count; t0 += gridDim.x * (2 * kThreads)) {
  float4 O0[2], O1[2]; bool mine[2]; unsigned bins[2]; uint32_t cols[2];
#pragma unroll
  for (int rep = 0; rep < 2; ++rep) {
  const unsigned t = t0 + rep * kThreads + threadIdx.x;
  const bool live = t < a.count;
  bool pass = false;
  float4 o0 = make_float4(0.f, 0.f, 0.f, 0.f), o1 = o0;
  int ptype = 0;
  unsigned bin = 0u;
  uint32_t com_col = 0u;
  if (live) {
    const unsigned long long h = history_of(a.first + t, a.perm_a, a.n_total);
    // group of h: last g with off[g] <= h (empty groups have off[g] == off[g+1] and are skipped by "last")
    if (a.perm_a == 0 && g >= 0) {
      while (g + 1 < m.n_groups && s_off[g + 1] <= h) ++g;
    } else {
      int lo = 0, hi = m.n_groups;         // invariant: off[lo] <= h < off[hi]
      while (hi - lo > 1) { int mid = (lo + hi) >> 1; if (s_off[mid] <= h) lo = mid; else hi = mid; }
      g = lo;
    }
    const int stype = (g >= m.n_ebin) + (g >= 2 * m.n_ebin), ebin = g - stype * m.n_ebin;     // three sub-sources
    ptype = m.particle_type[stype];
    Rng rng; rng.init(h, 0u, 0u);
    uint32_t x0, x1, x2, x3, y0, y1, y2, y3;
    rng.gen(a.ks, 0u, x0, x1, x2, x3);
    rng.gen(a.ks, 1u, y0, y1, y2, y3);
    // 1. let through the alias table
    const unsigned long long mm = (unsigned long long)x0 * m.n_let[g];
    const uint32_t col = (uint32_t)(mm >> 32), frac = (uint32_t)mm;
    const AliasEntry e = m.table[m.let_off[g] + col];
    const bool own = frac < e.thresh;
    const float ring = (float)(own ? e.ring_c : e.ring_a), sector = (float)(own ? e.sector_c : e.sector_a);
    // 2. position uniform in the let's area
    float sn, cs, px, py;
    const float pz = m.z_phsp;
    if (m.let_mode == 0) {
      const float r0 = ring * m.ring_width, r1 = (ring + 1.0f) * m.ring_width;
      const float r = sqrtf(r0 * r0 + u_co(x1) * (r1 * r1 - r0 * r0));
      sincospif(2.0f * (sector + u_co(x2)) * m.inv_nsec, &sn, &cs);
      px = r * cs; py = r * sn;
    } else {                                 // square let (Xbin, Ybin) = (ring, sector) fields of the entry
      px = m.grid_x0 + (ring + u_co(x1)) * m.let_size;
      py = m.grid_x0 + (sector + u_co(x2)) * m.let_size;
    }
    if (a.p2) {                                // the PSR this particle is from: one column per photon PSR, one per electron energy bin
      const int pr = m.let_mode == 0 ? (int)ring : min((int)(sqrtf(__fmaf_rn(px, px, py * py)) / m.ring_width), m.n_ring - 1);
      com_col = ptype == 0 ? (uint32_t)((stype * m.n_ebin + ebin) * m.n_ring + pr) : (uint32_t)(2 * m.n_ebin * m.n_ring + ebin);
    }
    // 3. energy uniform in the bin
    const float E = (m.e_min + (float)ebin * m.e_bin_width) + u_oc(x3) * m.e_bin_width;
    float dx, dy, dz;
    if (m.dir_K[stype] > 0) {
      // S4 / S5: direction from the Gaussian mixture of the PSR the position falls in (Eq. 6 / Eq. 7)
      const int K = m.dir_K[stype];
      const float r2 = __fmaf_rn(px, px, py * py), ir = rsqrtf(fmaxf(r2, 1e-30f)), r = r2 * ir;
      // ring of the position: for sector lets it is the let's own ring (an integer: no fp32 floor decision)
      const int i = m.let_mode == 0 ? (int)ring : min((int)(r / m.ring_width), m.n_ring - 1);
      const float4 *tab = m.dir_tab[stype] + ((size_t)ebin * m.n_ring + i) * K;
      const float tq = u_co(y0);
      int k = 0;
      float4 c = __ldg(tab);
      while (k < K - 1 && tq >= c.x) { ++k; c = __ldg(tab + k); }             // sequential search of P_{i,k}
      const float rho_n = sqrtf(-2.0f * logf(u_oc(y1)));
      sincospif(2.0f * u_co(y2), &sn, &cs);
      const float alpha = fminf(1.5f, fmaxf(-1.5f, __fmaf_rn(c.z * rho_n, cs, c.y)));
      const float beta = fminf(1.5f, fmaxf(-1.5f, c.w * rho_n * sn));
      float ul = tanf(alpha), vl = tanf(beta);
      const float inl = rsqrtf(__fmaf_rn(ul, ul, __fmaf_rn(vl, vl, 1.0f)));
      ul *= inl; vl *= inl;
      const float ct = r2 > 0.0f ? px * ir : 1.0f, st = r2 > 0.0f ? py * ir : 0.0f;   // theta = atan2(y, x)
      dx = ul * ct - vl * st; dy = ul * st + vl * ct; dz = inl;
      const float xj = px + dx / dz * m.jaw_dzx, yj = py + dy / dz * m.jaw_dzy;
      pass = xj >= m.jx_lo && xj <= m.jx_hi && yj >= m.jy_lo && yj <= m.jy_hi;
    } else {
    // 4. source point on the sub-source's Gaussian (Eq. 4)
    // (SFU log / root / trig here: the source point only tilts the direction by rho / (z_p - z_s))
    const float rho = m.sigma_src[stype] * sqrt_fast(-2.0f * __logf(u_oc(y0)));
    __sincosf(__fmaf_rn(6.283185307f, u_co(y1), -3.141592654f), &sn, &cs); sn = -sn; cs = -cs;
    (void)y2; (void)y3;
    const float qx = rho * cs, qy = rho * sn, qz = m.z_src[stype];
    // 5. direction (Eq. 5)
    dx = px - qx; dy = py - qy; dz = pz - qz;
    const float il = rsqrtf(dx * dx + dy * dy + dz * dz);
    dx *= il; dy *= il; dz *= il;
    // 6. thin-jaw test
    const float xj = qx + (px - qx) * m.jaw_tx[stype], yj = qy + (py - qy) * m.jaw_ty[stype];
    pass = xj >= m.jx_lo && xj <= m.jx_hi && yj >= m.jy_lo && yj <= m.jy_hi;
    }
    // 7. beam set-up
    const float *R = a.beam.R;
    const float bz = pz - a.beam.sad;
    o0.x = __fmaf_rn(R[0], px, __fmaf_rn(R[1], py, __fmaf_rn(R[2], bz, a.beam.iso[0])));
    o0.y = __fmaf_rn(R[3], px, __fmaf_rn(R[4], py, __fmaf_rn(R[5], bz, a.beam.iso[1])));
    o0.z = __fmaf_rn(R[6], px, __fmaf_rn(R[7], py, __fmaf_rn(R[8], bz, a.beam.iso[2])));
    o0.w = E;
    o1.x = __fmaf_rn(R[0], dx, __fmaf_rn(R[1], dy, R[2] * dz));
    o1.y = __fmaf_rn(R[3], dx, __fmaf_rn(R[4], dy, R[5] * dz));
    o1.z = __fmaf_rn(R[6], dx, __fmaf_rn(R[7], dy, R[8] * dz));
    const unsigned long long qE = (unsigned long long)quanta(E);
    q_inc += qE;
    if (!pass) {
      q_jaw += qE;
      if (a.fp) {
        Fnv f; f.init(0u); f.byte('J');
        atomicAdd(a.fp + (h - a.fp_base), f.v);
      }
    } else if (a.compact) {
      // P4 entry: a particle that starts outside the grid is moved to its entry point (+ eps); a miss ends here
      int vi, vj, vk;
      if (!locate(a.g, o0.x, o0.y, o0.z, vi, vj, vk) && !enter(a.g, o0.x, o0.y, o0.z, o1.x, o1.y, o1.z, vi, vj, vk)) {
        ++n_miss; pass = false; q_esc += qE;
        if (a.fp) {
          Fnv f; f.init(0u);
          if (ptype) f.u32(0u);           // an electron track records its (zero) step count first
          f.byte('M');
          atomicAdd(a.fp + (h - a.fp_base), f.v);
        }
      } else if (tiles) bin = tile_bin(a.tm, vi, vj, vk);
    }
  }
  if (a.compact) {
    o1.w = __uint_as_float(t | ((unsigned)ptype << 31));
    O0[rep] = o0; O1[rep] = o1; mine[rep] = live && pass; bins[rep] = bin; cols[rep] = com_col;
  } else if (live) {
    o1.w = pass ? (float)g : -(float)g - 1.0f;
    a.p0[t] = o0; a.p1[t] = o1;
  }
  }
  if (a.compact) {
    // survivors of both histories packed with ONE queue-tail atomic per warp (deferring the stores behind the atomic's
    // latency was measured: no gain)
    const unsigned keep0 = __ballot_sync(kFull, mine[0]), keep1 = __ballot_sync(kFull, mine[1]);
    const unsigned n0 = __popc(keep0), tot = n0 + __popc(keep1);
    unsigned base = 0;
    if (lane == 0 && tot) base = atomicAdd(&a.ctl->n_pb, tot);
    base = __shfl_sync(kFull, base, 0);
#pragma unroll
    for (int rep = 0; rep < 2; ++rep)
      if (mine[rep]) {
        const unsigned dst = base + (rep ? n0 : 0u) + __popc((rep ? keep1 : keep0) & ((1u << lane) - 1u));
        __stcs(a.p0 + dst, O0[rep]); __stcs(a.p1 + dst, O1[rep]);         // write-once / read-once: streaming, keeps L2 for the phantom and the grid
        if (a.p2) a.p2[dst] = cols[rep];
        if (tiles) atomicAdd(&s_hist[bins[rep]], 1u);
      }
  }
  }
  // ledgers: incident, jaw-rejected and escaped (missed) energy, one 128-bit add per warp and ledger, spread over slots
  if (a.ctl) {
    q_inc = warp_sum_u64(q_inc); q_jaw = warp_sum_u64(q_jaw); q_esc = warp_sum_u64(q_esc);
    const unsigned nm = __reduce_add_sync(kFull, n_miss);
    if (lane == 0) {
      unsigned long long (*L)[2] = a.ctl->ledger[(blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5)) % kLedgerSlots];
      add128(L[0], q_inc); add128(L[3], q_jaw); add128(L[2], q_esc);
      if (nm) { atomicAdd(&a.ctl->n_missed, (unsigned long long)nm); if (a.stats) atomicAdd(&a.ctl->stat[ST_MISSED], (unsigned long long)nm); }
    }
  }
  if (tiles) {
    __syncthreads();
    for (int i = threadIdx.x; i < a.tm.nbins; i += kThreads) { const unsigned c = s_hist[i]; if (c) atomicAdd(a.tile_count + i, c); }
  }
}

// Counts → cursors (exclusive prefix sum over the bins, one CTA of 1024 threads), counts zeroed for the next batch.
__global__ void __launch_bounds__(1024) k_tile_scan(unsigned *count, unsigned *cursor, int nbins) {
  __shared__ unsigned s_w[32];
  const int per = (nbins + 1023) / 1024, b0 = threadIdx.x * per;
  unsigned loc[4], sum = 0;                                  // per <= 4 (kTileBinsMax / 1024)
#pragma unroll
  for (int k = 0; k < 4; ++k) { loc[k] = (k < per && b0 + k < nbins) ? count[b0 + k] : 0u; sum += loc[k]; }
  unsigned inc = sum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const unsigned v = __shfl_up_sync(kFull, inc, o); if ((threadIdx.x & 31) >= o) inc += v; }
  if ((threadIdx.x & 31) == 31) s_w[threadIdx.x >> 5] = inc;
  __syncthreads();
  if (threadIdx.x < 32) {
    unsigned w = s_w[threadIdx.x], wi = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const unsigned v = __shfl_up_sync(kFull, wi, o); if (threadIdx.x >= o) wi += v; }
    s_w[threadIdx.x] = wi - w;
  }
  __syncthreads();
  unsigned run = s_w[threadIdx.x >> 5] + inc - sum;
#pragma unroll
  for (int k = 0; k < 4; ++k) if (k < per && b0 + k < nbins) { cursor[b0 + k] = run; run += loc[k]; count[b0 + k] = 0u; }
}

// Moves the packed survivors (p planes) to their tile-ordered places (q planes).  A CTA takes chunks of kTileChunk
// particles: local histogram in shared memory, one global reservation per non-empty bin, then the moves.
constexpr int kTileChunk = 4096;
struct ScatterArgs {
  Grid g; TileMap tm;
  const float4 *p0, *p1; const uint32_t *p2;
  float4 *q0, *q1; uint32_t *q2;
  const unsigned *n_pb; unsigned *cursor;
};
__global__ void __launch_bounds__(kThreads) k_tile_scatter(const __grid_constant__ ScatterArgs a) {
  extern __shared__ unsigned s_t[];                          // [nbins] counts, then [nbins] bases
  unsigned *s_cnt = s_t, *s_base = s_t + a.tm.nbins;
  const unsigned n = *a.n_pb;
  for (unsigned c0 = blockIdx.x * kTileChunk; c0 < n; c0 += gridDim.x * kTileChunk) {
    for (int i = threadIdx.x; i < a.tm.nbins; i += kThreads) s_cnt[i] = 0u;
    __syncthreads();
    unsigned bins[kTileChunk / kThreads];
#pragma unroll
    for (int k = 0; k < kTileChunk / kThreads; ++k) {
      const unsigned i = c0 + k * kThreads + threadIdx.x;
      bins[k] = 0xffffffffu;
      if (i < n) {
        const float4 A = __ldcs(a.p0 + i);
        int vi, vj, vk; locate(a.g, A.x, A.y, A.z, vi, vj, vk);     // inside the grid: k_sample moved it to its entry point
        bins[k] = tile_bin(a.tm, vi, vj, vk);
        atomicAdd(&s_cnt[bins[k]], 1u);
      }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < a.tm.nbins; i += kThreads) { const unsigned c = s_cnt[i]; if (c) s_base[i] = atomicAdd(a.cursor + i, c); s_cnt[i] = 0u; }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kTileChunk / kThreads; ++k) {
      const unsigned i = c0 + k * kThreads + threadIdx.x;
      if (bins[k] != 0xffffffffu) {
        const unsigned dst = s_base[bins[k]] + atomicAdd(&s_cnt[bins[k]], 1u);
        __stcs(a.q0 + dst, __ldcs(a.p0 + i)); __stcs(a.q1 + dst, __ldcs(a.p1 + i));
        if (a.p2) a.q2[dst] = a.p2[i];
      }
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------ small helpers
// Folds the finished batch's counters into the per-call totals and resets them.
__global__ void k_next_batch(Control *c) {
  c->n_accepted += c->n_pb;
  c->hw_eq = max(c->hw_eq, c->n_eq);
  c->n_pb = c->head_pb = c->n_eq = c->head_eq = c->head_pb_e = 0;
}

// Packs the caller's phantom into one 32-bit word per voxel (density rounded to nearest on a 22-bit
// mantissa, material in the two low bits) and finds the largest PACKED density per material (Woodcock
// majorant input).  Densities are >= 0, so float order = uint order.
__global__ void k_pack_phantom(const float *density, const uint8_t *material, size_t n, uint32_t *vox, Control *c) {
  float best[3] = {0.f, 0.f, 0.f};
  for (size_t v = blockIdx.x * (size_t)blockDim.x + threadIdx.x; v < n; v += (size_t)gridDim.x * blockDim.x) {
    const uint32_t bits = (__float_as_uint(density[v]) + 2u) & ~3u; const int mt = min((int)material[v], 2);
    vox[v] = bits | (uint32_t)mt;
    const float d = __uint_as_float(bits);
    if (mt == 0) best[0] = fmaxf(best[0], d); else if (mt == 1) best[1] = fmaxf(best[1], d); else best[2] = fmaxf(best[2], d);
  }
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    float b = best[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) b = fmaxf(b, __shfl_xor_sync(kFull, b, o));
    if ((threadIdx.x & 31) == 0 && b > 0.f) atomicMax((unsigned *)&c->rhomax[k], __float_as_uint(b));
  }
}

// One bit per voxel: com_index[v] != 0 (the commissioning tally's measurement voxels are few: PAPER.md:134).
// `coarse` (zeroed before): one bit per 512 consecutive voxels = 16 words of `mask`.
__global__ void k_com_mask(const int *com_index, size_t n, uint32_t *mask, uint32_t *coarse) {
  const size_t w = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
  if (w * 32 >= n) return;
  uint32_t m = 0u;
  for (int b = 0; b < 32 && w * 32 + b < n; ++b) m |= (com_index[w * 32 + b] != 0 ? 1u : 0u) << b;
  mask[w] = m;
  if (m) atomicOr(coarse + (w >> 9), 1u << ((w >> 4) & 31));
}

// "All words of the 4x4x4 cell at (ci, cj, ck) of an array of (n0, n1, n2) words equal w0" - rows of four words are read as
// one 16-byte load when they are aligned (n0 a multiple of 4) and the cell is not clipped in x.
__device__ __forceinline__ bool cell_uniform(const uint32_t *w, int n0, int n1, int n2, int ci, int cj, int ck, uint32_t w0) {
  bool uni = true;
  const bool vec = (n0 & 3) == 0;                              // (then ci*4 + 4 <= n0 as well)
  for (int k = ck * 4; k < min(ck * 4 + 4, n2); ++k)
    for (int j = cj * 4; j < min(cj * 4 + 4, n1); ++j) {
      const size_t row = ((size_t)k * n1 + j) * n0 + ci * 4;
      if (vec) { const uint4 q = *reinterpret_cast<const uint4 *>(w + row); uni &= q.x == w0 && q.y == w0 && q.z == w0 && q.w == w0; }
      else for (int i = 0; i < min(4, n0 - ci * 4); ++i) uni &= w[row + i] == w0;
    }
  return uni;
}

// The brick table of the hierarchical phantom (Grid::brick): one thread per brick of 4x4x4 voxels (clipped at the grid's edge).
__global__ void k_bricks(const uint32_t *vox, int nx, int ny, int nz, int nbx, int nby, unsigned nbricks, uint32_t *brick, Control *c) {
  const unsigned b = blockIdx.x * blockDim.x + threadIdx.x;
  bool uni = false;
  if (b < nbricks) {
    const int bi = (int)(b % (unsigned)nbx), bj = (int)((b / (unsigned)nbx) % (unsigned)nby), bk = (int)(b / ((unsigned)nbx * (unsigned)nby));
    const uint32_t w0 = vox[((size_t)(bk * 4) * ny + bj * 4) * nx + bi * 4];
    uni = cell_uniform(vox, nx, ny, nz, bi, bj, bk, w0);
    brick[b] = uni ? (w0 | 0x80000000u) : 0u;
  }
  const unsigned n = __popc(__ballot_sync(kFull, uni));
  if ((threadIdx.x & 31) == 0 && n) atomicAdd(&c->n_uniform_bricks, n);
}

// The super-brick table on top of it: one thread per super-brick of 4x4x4 bricks (clipped at the edge).
__global__ void k_sbricks(const uint32_t *brick, int nbx, int nby, int nbz, int nsx, int nsy, unsigned nsb, uint32_t *sbrick, Control *c) {
  const unsigned b = blockIdx.x * blockDim.x + threadIdx.x;
  bool uni = false;
  if (b < nsb) {
    const int si = (int)(b % (unsigned)nsx), sj = (int)((b / (unsigned)nsx) % (unsigned)nsy), sk = (int)(b / ((unsigned)nsx * (unsigned)nsy));
    const uint32_t w0 = brick[((size_t)(sk * 4) * nby + sj * 4) * nbx + si * 4];
    uni = (w0 & 0x80000000u) != 0u && cell_uniform(brick, nbx, nby, nbz, si, sj, sk, w0);
    sbrick[b] = uni ? w0 : 0u;
  }
  const unsigned n = __popc(__ballot_sync(kFull, uni));
  if ((threadIdx.x & 31) == 0 && n) atomicAdd(&c->n_uniform_sbricks, n);
}

// Photon cross-section data: layout in pslmc_device.cuh (XsTable), evaluated in double.  The sigma_KN nodes depend on
// the energy range only and are built once per psl_t; the majorant head needs the phantom's rhomax (c, may be null).
__global__ void k_build_xs(const Control *c, float *data, double x0, double h, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (c && i < 3) {                               // (k_photon recomputes this head per CTA from the call's rhomax; mc_xs_debug reads it here)
    const double rm = (double)c->rhomax[i];
    data[4 * i] = (float)(rm * (double)c_mat.ne[i]); data[4 * i + 1] = (float)(rm * (double)c_mat.cphoto[i]);
    data[4 * i + 2] = (float)(rm * (double)c_mat.ppair[i]); data[4 * i + 3] = 0.0f;
  }
  if (i > n) return;
  const double E = exp2(x0 + h * (double)i);
  const double al = E / kMeD, L = log1p(2.0 * al), t = 1.0 + 2.0 * al;
  const double skn = kTwoPiRe2 * ((1.0 + al) / (al * al) * (2.0 * (1.0 + al) / t - L / al) + L / (2.0 * al) - (1.0 + 3.0 * al) / (t * t));
  data[kXsHead + i] = (float)skn;
}

// Parity probe: the table lookup k_photon does, for a list of energies.  out: (sigma_KN, ln^2(E/1.022), mu_max) per energy.
__global__ void k_xs_debug(XsTable xs, const float *E, size_t n, float *out) {
  const size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  float skn, ie3, lp2, mu;
  xs_lookup(xs.data, xs.x0, xs.inv_h, xs.n, E[i], skn, ie3, lp2, mu);
  out[3 * i] = skn; out[3 * i + 1] = lp2; out[3 * i + 2] = mu;
}

// dose[v] = acc[v] 2^-32 / (rho_v V N).  Deposits are never negative, so a negative accumulator has wrapped past
// 2^63 quanta (2.1e9 MeV in one voxel): flagged, mc_dose then returns MC_E_OVERFLOW.  dose == nullptr: scan only.
__global__ void k_finalise(const long long *acc, const float *density, size_t n, double inv_vn, double *dose, Control *c) {
  bool wrapped = false;
  for (size_t v = blockIdx.x * (size_t)blockDim.x + threadIdx.x; v < n; v += (size_t)gridDim.x * blockDim.x) {
    const long long q = acc[v];
    wrapped |= q < 0;
    if (dose) { const float rho = density[v]; dose[v] = rho > 0.f ? (double)q * (1.0 / 4294967296.0) * inv_vn / (double)rho : 0.0; }
  }
  if (wrapped) atomicOr(&c->overflow, 2u);
}

__global__ void k_philox_debug(unsigned long long seed, unsigned long long h, uint32_t track, uint32_t block, uint32_t *out) {
  uint32_t ks[20];
  for (int r = 0; r < 10; ++r) { ks[2 * r] = (uint32_t)seed + (uint32_t)r * 0x9E3779B9u; ks[2 * r + 1] = (uint32_t)(seed >> 32) + (uint32_t)r * 0xBB67AE85u; }
  Rng r; r.init(h, track, 0u);
  r.gen(ks, block, out[0], out[1], out[2], out[3]);
}

}  // namespace pslmc
