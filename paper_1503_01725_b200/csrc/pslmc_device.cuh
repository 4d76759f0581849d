// pslmc_device.cuh — device-side building blocks of libpslmc (sm_100a): counter-based RNG,
// physics in fp32, geometry, int64 fixed-point scoring.  Definitions: DESIGN.md R1, P1-P9, S1, F1.
// Shares nothing with oracle/ (which is test infrastructure); constants are typed here on their own.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace pslmc {

// ------------------------------------------------------------------ model constants
constexpr float  kMe      = 0.51099895f;      // electron rest energy (MeV)
constexpr double kMeD     = 0.51099895;
constexpr double kTwoPiRe2 = 2.0 * 3.14159265358979323846 * 7.940787e-26;   // 2 pi r_e^2 (cm^2)
constexpr float  kEPair   = 1.022f;           // pair threshold / annihilation total (MeV)
constexpr float  kEAnnih  = 0.511f;
constexpr float  kPcut    = 0.05f;            // photon cut-off
constexpr float  kEcut    = 0.2f;             // electron cut-off
constexpr float  kEpsB    = 1e-4f;            // boundary nudge (cm)
constexpr float  kFe      = 0.12f;            // energy-loss fraction per condensed-history step
constexpr float  kPi      = 3.14159265358979323846f;

struct Materials {       // index: 0 water, 1 lung, 2 bone
  float ne[3];           // electrons per gram
  float cphoto[3];       // cm^2 g^-1 MeV^3
  float ppair[3];        // cm^2 g^-1
  float sscale[3];       // stopping-power scale
  float inv_x0[3];       // 1 / radiation length (cm^2/g)
};
__constant__ Materials c_mat = {
    {3.343e23f, 3.343e23f, 3.100e23f},
    {2.77e-6f, 2.77e-6f, 2.2e-5f},
    {9.6e-4f, 9.6e-4f, 1.3e-3f},
    {1.0f, 1.0f, 0.92f},
    {1.0f / 36.08f, 1.0f / 36.08f, 1.0f / 27.2f}};

// ------------------------------------------------------------------ R1: Philox4x32-10
// The stream of a track (R1): blocks 0, 1, 2, ... of Philox4x32-10 keyed by the seed with counter
// (block, track, history lo, history hi).  Every event takes the next whole block, so an event site is one
// unconditional generation for all its lanes and the per-lane state is just the block counter.  ks = the 10
// round keys (k0 + r*0x9E3779B9, k1 + r*0xBB67AE85), host-computed kernel parameters: the XORs take them straight
// from the constant bank.
struct Rng {
  uint32_t track, hlo, hhi, blk;
  __device__ __forceinline__ void init(uint64_t h, uint32_t trk, uint32_t first_block) {
    hlo = (uint32_t)h; hhi = (uint32_t)(h >> 32); track = trk; blk = first_block;
  }
  __device__ __forceinline__ void gen(const uint32_t (&ks)[20], uint32_t j, uint32_t &g0, uint32_t &g1, uint32_t &g2, uint32_t &g3) const {
    uint32_t x0 = j, x1 = track, x2 = hlo, x3 = hhi;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
      const uint32_t h0 = __umulhi(0xD2511F53u, x0), l0 = 0xD2511F53u * x0;
      const uint32_t h1 = __umulhi(0xCD9E8D57u, x2), l1 = 0xCD9E8D57u * x2;
      x0 = h1 ^ x1 ^ ks[2 * r]; x1 = l1; x2 = h0 ^ x3 ^ ks[2 * r + 1]; x3 = l0;
    }
    g0 = x0; g1 = x1; g2 = x2; g3 = x3;
  }
  __device__ __forceinline__ void next(const uint32_t (&ks)[20], uint32_t &g0, uint32_t &g1, uint32_t &g2, uint32_t &g3) {
    gen(ks, blk, g0, g1, g2, g3); ++blk;
  }
};

__device__ __forceinline__ float u_co(uint32_t x) { return (float)(x >> 8) * (1.0f / 16777216.0f); }          // [0,1)
__device__ __forceinline__ float u_oc(uint32_t x) { return (float)((x >> 8) + 1u) * (1.0f / 16777216.0f); }   // (0,1]

__device__ __forceinline__ uint32_t child_track(uint32_t parent, uint32_t n, uint32_t c) {
  return (((parent ^ 0x9E3779B9u) * 0x01000193u) ^ ((n << 2) | c)) * 0x01000193u;
}

// ------------------------------------------------------------------ F1: FNV-1a-64
struct Fnv {
  uint64_t v;
  __device__ __forceinline__ void init(uint32_t track) { v = 0xcbf29ce484222325ull; u32(track); }
  __device__ __forceinline__ void byte(uint32_t b) { v = (v ^ (uint64_t)b) * 0x100000001b3ull; }
  __device__ __forceinline__ void u32(uint32_t x) { byte(x & 255u); byte((x >> 8) & 255u); byte((x >> 16) & 255u); byte(x >> 24); }
};

// ------------------------------------------------------------------ phantom + scoring
struct Grid {
  int nx, ny, nz;
  float ox, oy, oz, dx, dy, dz, idx, idy, idz;      // origin, voxel size, reciprocal voxel size
  const float   *density;                            // caller's arrays (k_pack_phantom, k_finalise)
  const uint8_t *material;
  const uint32_t *vox;                               // packed phantom, one gather per voxel: density bits rounded to a
                                                     // 22-bit mantissa | material index in the two low bits
  // Hierarchical phantom: one word per brick of 4x4x4 voxels = the brick's common voxel word | 0x80000000 when all its
  // voxels are equal (densities are >= 0, so bit 31 of a voxel word is free), else 0; and the same once more per
  // super-brick of 4x4x4 bricks (16^3 voxels).  A phantom that is mostly uniform super-bricks (water tanks: >= 90 %,
  // decided per call on the device) is then read top down: the super-brick table (16 KiB for 256^3 voxels:
  // L1-resident), the brick table (L2) where a super-brick is mixed, the 4-byte-per-voxel array only where a brick is
  // mixed.
  const uint32_t *brick, *sbrick; const unsigned *n_uniform, *n_uniform_sb; int nbx, nby, nsx, nsy; unsigned nbricks, nsbricks;
  unsigned long long *acc;                           // int64 fixed-point dose accumulator (2^-32 MeV)
  // commissioning tally, off when com_index is null: com_index[v] = 0 or 1 + row,
  // com_dose[col * com_rows + row], col = the PSR unit the history was sampled from
  const int *com_index; unsigned long long *com_dose; int com_rows;
  const uint32_t *com_mask, *com_coarse;             // one bit per voxel: com_index[v] != 0, and one bit per 512 consecutive voxels: any of
                                                     // them (built per call; the coarse map stays in L1, the index array is read only on a hit)
};

__device__ __forceinline__ long long quanta(float e) { return __float2ll_rn(e * 4294967296.0f); }

__device__ __forceinline__ bool locate(const Grid &g, float x, float y, float z, int &i, int &j, int &k) {
  float fi = floorf((x - g.ox) * g.idx), fj = floorf((y - g.oy) * g.idy), fk = floorf((z - g.oz) * g.idz);
  bool in = fi >= 0.0f && fi < (float)g.nx && fj >= 0.0f && fj < (float)g.ny && fk >= 0.0f && fk < (float)g.nz;
  i = (int)fi; j = (int)fj; k = (int)fk;
  return in;
}
// true: read the phantom top down through the super-brick and brick tables; false: read the per-voxel array directly
// (a mixed cell costs one more dependent read per level, so the tables are used when >= 90 % of the super-bricks are uniform)
__device__ __forceinline__ bool use_bricks(const Grid &g) { return g.brick != nullptr && *g.n_uniform_sb * 10ull >= g.nsbricks * 9ull; }
__device__ __forceinline__ void fetch_voxel(const Grid &g, bool bricks, int i, int j, int k, int v, float &rho, int &mt) {
  uint32_t p = 0u;
  if (bricks) {
    p = __ldg(g.sbrick + ((i >> 4) + g.nsx * ((j >> 4) + g.nsy * (k >> 4))));
    if (!(p & 0x80000000u)) p = __ldg(g.brick + ((i >> 2) + g.nbx * ((j >> 2) + g.nby * (k >> 2))));
  }
  if (p & 0x80000000u) p &= 0x7fffffffu; else p = __ldg(g.vox + v);
  rho = __uint_as_float(p & ~3u); mt = (int)(p & 3u);
}
__device__ __forceinline__ int vox_index(const Grid &g, int i, int j, int k) { return (k * g.ny + j) * g.nx + i; }

// Ray/box entry for a track that starts outside the grid.  false = misses the phantom.
__device__ __forceinline__ bool enter(const Grid &g, float &x, float &y, float &z, float u, float v, float w,
                                      int &i, int &j, int &k) {
  const float lo[3] = {g.ox, g.oy, g.oz};
  const float hi[3] = {g.ox + g.nx * g.dx, g.oy + g.ny * g.dy, g.oz + g.nz * g.dz};
  const float p[3] = {x, y, z}, d[3] = {u, v, w};
  float tmin = -INFINITY, tmax = INFINITY;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    if (d[a] == 0.0f) { if (p[a] < lo[a] || p[a] >= hi[a]) return false; continue; }
    float t1 = (lo[a] - p[a]) / d[a], t2 = (hi[a] - p[a]) / d[a];      // IEEE division: the entry point seeds every later voxel decision
    tmin = fmaxf(tmin, fminf(t1, t2)); tmax = fminf(tmax, fmaxf(t1, t2));
  }
  if (tmin > tmax || tmax <= 0.0f) return false;
  float s = fmaxf(tmin, 0.0f) + kEpsB;
  x += s * u; y += s * v; z += s * w;
  return locate(g, x, y, z, i, j, k);
}

// ------------------------------------------------------------------ physics
__device__ __forceinline__ float rcp_fast(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

// Photon cross-section data (built per mc_dose call on the device, in double, by k_build_xs), kept in shared
// memory by k_photon:  floats [0,12) = per material m the Woodcock majorant coefficients
// (rhomax_m ne_m, rhomax_m cphoto_m, rhomax_m ppair_m, 0);  floats [12, 12 + n + 1) = sigma_KN at
// log2(E) = x0 + i*h, interpolated linearly (relative error ~1e-7 at n = 4096: DESIGN.md §6).  1/E^3 and
// ln(E/1.022) are computed directly (the latter from the same log2 E), so
// mu_max = max_m (A_m sigma_KN + B_m / E^3 + C_m ln^2) carries no interpolation error of its own.
constexpr int kXsHead = 12;
struct XsTable { const float *data; float x0, inv_h; int n; };      // n intervals, n + 1 nodes after the head

__device__ __forceinline__ void xs_lookup(const float *tab, float x0, float inv_h, int n, float E,
                                          float &skn, float &inv_e3, float &lp2, float &mu_max) {
  const float lg = __log2f(E);
  float t = (lg - x0) * inv_h;
  t = fminf(fmaxf(t, 0.0f), (float)n);
  const int i = min((int)t, n - 1);
  const float f = t - (float)i;
  const float a = tab[kXsHead + i], b = tab[kXsHead + i + 1];
  skn = __fmaf_rn(f, b - a, a);
  const float l = E > kEPair ? (lg - 0.03139551f) * 0.69314718f : 0.0f;      // log2(1.022) = 0.0313955
  lp2 = l * l;
  inv_e3 = rcp_fast(E * E * E);
  const float4 *mj = reinterpret_cast<const float4 *>(tab);
  float m = 0.0f;
#pragma unroll
  for (int k = 0; k < 3; ++k) { const float4 c = mj[k]; m = fmaxf(m, __fmaf_rn(c.x, skn, __fmaf_rn(c.y, inv_e3, c.z * lp2))); }
  mu_max = m;
}

__device__ __forceinline__ float sqrt_fast(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

__device__ __forceinline__ void rotate(float &u, float &v, float &w, float ct, float st, float uphi) {
  float sp, cp;
  // azimuth 2 pi uphi through the SFU on an argument in [-pi, pi): sin/cos(phi) = -sin/cos(phi - pi);
  // absolute error ~4e-7, measured effect on the oracle-identical fraction < 1e-5
  __sincosf(__fmaf_rn(6.283185307f, uphi, -3.141592654f), &sp, &cp); sp = -sp; cp = -cp;
  float nx, ny, nz;
  const float s2 = __fmaf_rn(u, u, v * v);                // = 1 - w^2 for a unit vector, without the cancellation
  if (s2 > 1e-20f) {
    const float is = rsqrtf(s2), s = s2 * is, a = st * is;
    nx = __fmaf_rn(u, ct, a * __fmaf_rn(u * w, cp, -(v * sp)));
    ny = __fmaf_rn(v, ct, a * __fmaf_rn(v * w, cp, u * sp));
    nz = __fmaf_rn(w, ct, -(s * st) * cp);
  } else {
    nx = st * cp; ny = st * sp; nz = w > 0.0f ? ct : -ct;
  }
  const float inv = rsqrtf(__fmaf_rn(nx, nx, __fmaf_rn(ny, ny, nz * nz)));
  u = nx * inv; v = ny * inv; w = nz * inv;
}

// ------------------------------------------------------------------ warp helpers
__device__ __forceinline__ unsigned long long warp_sum_u64(unsigned long long v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
// Warp sum of energy quanta known to be < 2^44 each (E < 4096 MeV): two hardware integer reductions
// on the low 22 and the high 22 bits (exact).
__device__ __forceinline__ unsigned long long warp_sum_q(unsigned long long v) {
  const unsigned lo = __reduce_add_sync(0xffffffffu, (unsigned)v & 0x3fffffu);
  const unsigned hi = __reduce_add_sync(0xffffffffu, (unsigned)(v >> 22));
  return ((unsigned long long)hi << 22) + lo;
}
// 128-bit unsigned accumulate into (lo, hi) words in global memory.
__device__ __forceinline__ void add128(unsigned long long *lohi, unsigned long long q) {
  if (q == 0) return;
  unsigned long long old = atomicAdd(lohi, q);
  if (old + q < old) atomicAdd(lohi + 1, 1ull);
}

}  // namespace pslmc
