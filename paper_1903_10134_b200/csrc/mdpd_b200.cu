// mdpd_b200.cu -- hand-written CUDA (sm_100a) for one mDPD velocity-Verlet timestep + the C-ABI of include/mdpd.h.
//
// Paper: arxiv/paper_1903_10134.  Eq. (1) and the weight functions: PAPER.md L75-81; Algorithm 1
// (x -> rho -> f -> v): PAPER.md L125-133; body force: L186; frozen walls: L162.  Readings R1..R18 and the hash
// specification: DESIGN.md sections 3 and 4.  This file shares nothing with oracle/ (the fp64 CPU oracle).
//
// Device state: pos float4 = (x, y, z, bits(tag | type << 31)), vel float4 = (vx, vy, vz, rho),
// both double-buffered for the Morton counting sort; force float4; xbuild float4 (positions at the last list build);
// Verlet list split in a near part (r < rd + skin at build: all the density pass needs) and a far part, both stored
// column-major ([k][i]) so that a warp reads consecutive i at fixed k in one coalesced request.
#include "mdpd.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

namespace {

constexpr unsigned ERR_OVERFLOW = 1u;
constexpr unsigned ERR_NAN = 2u;
constexpr int TPB = 128;           // threads per block of the per-particle kernels
constexpr int SCAN_TPB = 256;      // scan: 256 threads x 8 items
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = SCAN_TPB * SCAN_ITEMS;

// Device-resident control block: everything that changes from step to step lives here, so that the kernel arguments
// of a step are constant (CUDA-graph friendly) and no host round trip is needed for the rebuild decision.
struct Ctl {
  unsigned cur;       // index of the live pos/vel buffer
  unsigned rebuild;   // 1: the rebuild chain of this step runs (src = cur ^ 1, dst = cur)
  unsigned maxdisp2;  // float bits of the largest squared displacement since the last build
  unsigned ticket;    // last-block-done counter of k_integrate
  unsigned step;      // index k of the time level of the last force evaluation (hash input)
  unsigned err;       // ERR_* bits, latched
  unsigned max_nbr;   // longest list at the last build
  unsigned pair_count_lo;
  unsigned long long steps, rebuilds, bounces, sum_nbr, overflow, nan_events, pair_count, sum_near;
};

struct DevP {  // passed by value to every kernel
  // arrays
  float4* pos[2];
  float4* vel[2];
  float4* force;
  float4* xbuild;
  unsigned* cell_rank;   // [ncell] linear cell -> Morton rank
  unsigned* cell_count;  // [ncell] histogram (self-cleaning)
  unsigned* cell_start;  // [ncell + 1]
  unsigned* scan_bsum;   // [nblocks of the scan]
  unsigned* pcell;       // [N] Morton rank of the particle's cell (old order)
  unsigned* order;       // [N] old index of the particle that goes to sorted slot s (unordered inside a cell)
  unsigned* nbr_near;    // [cap_near][N]
  unsigned* nbr_far;     // [cap_far][N]
  unsigned* nnbr;        // [N] near | far << 16
  const unsigned char* mask;
  Ctl* ctl;
  // sizes
  unsigned N, ncell, cap_near, cap_far;
  int ncx, ncy, ncz;
  int mx, my, mz;
  // geometry
  float Lx, Ly, Lz;
  float icx, icy, icz;  // 1 / cell edge
  float inv_voxel;
  float rlist2, rnear2, rc2, rd2;
  float margin;  // particles farther than this from every box face need no minimum-image test
  // physics
  float inv_rc, inv_rd, Krho;
  float A, B, gamma, sig_c;  // sig_c = sigma * sqrt(3) * 2^-23 / sqrt(dt)
  float dt, hdt_m;           // dt, 0.5 dt / m
  float fgx, fgy, fgz;       // m g
  float thr2;                // (skin / 2)^2
  unsigned seed;
};

__device__ __forceinline__ unsigned f2u(float f) { return __float_as_uint(f); }
__device__ __forceinline__ float u2f(unsigned u) { return __uint_as_float(u); }

__device__ __forceinline__ float minimg(float d, float L) {
  const float h = 0.5f * L;
  if (d > h) d -= L;
  else if (d < -h) d += L;
  return d;
}

__device__ __forceinline__ float wrap1(float x, float L) {  // |x - [0,L)| << L here (one step of drift)  R12
  if (x >= L) x -= L;
  else if (x < 0.0f) x += L;
  if (x >= L) x = 0.0f;
  return x;
}

__device__ __forceinline__ int cell_coord(float x, float inv_edge, int nc) {
  int c = (int)(x * inv_edge);
  return min(max(c, 0), nc - 1);
}

// ----------------------------------------------------------------------------------------------------------------
// Pair hash, DESIGN.md section 4 (restated from that text).  Round keys depend on (step, seed) only.
// ----------------------------------------------------------------------------------------------------------------
struct HashKeys {
  unsigned k[6];
};
__device__ __forceinline__ HashKeys make_keys(unsigned step, unsigned seed) {
  HashKeys K;
  K.k[0] = step;
  K.k[1] = seed;
  K.k[2] = step + 0x9E3779B9u;
  K.k[3] = seed + 0xBB67AE85u;
  K.k[4] = step + 2u * 0x9E3779B9u;
  K.k[5] = seed + 2u * 0xBB67AE85u;
  return K;
}
__device__ __forceinline__ unsigned pair_hash(unsigned a, unsigned b, const HashKeys& K) {
  unsigned x = min(a, b), y = max(a, b);
#pragma unroll
  for (int r = 0; r < 6; ++r) {
    unsigned long long p = (unsigned long long)0xD256D193u * (unsigned long long)x;
    unsigned hi = (unsigned)(p >> 32), lo = (unsigned)p;
    x = hi ^ y ^ K.k[r];
    y = lo;
  }
  return x;
}

// ----------------------------------------------------------------------------------------------------------------
// load / unload
// ----------------------------------------------------------------------------------------------------------------
__global__ void k_pack(DevP p, const float* __restrict__ pos, const float* __restrict__ vel,
                       const unsigned char* __restrict__ type, unsigned buf) {
  unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.N) return;
  unsigned t = type ? (type[i] != 0) : 0u;
  float x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
  // general wrap at load time (inputs may be anywhere): x - L floor(x / L), result == L -> 0   (R12)
  x -= p.Lx * floorf(x / p.Lx);
  y -= p.Ly * floorf(y / p.Ly);
  z -= p.Lz * floorf(z / p.Lz);
  if (!(x < p.Lx)) x = 0.0f;
  if (!(y < p.Ly)) y = 0.0f;
  if (!(z < p.Lz)) z = 0.0f;
  if (x < 0.0f) x = 0.0f;
  if (y < 0.0f) y = 0.0f;
  if (z < 0.0f) z = 0.0f;
  p.pos[buf][i] = make_float4(x, y, z, u2f(i | (t << 31)));
  float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
  if (!t) {
    v.x = vel[3 * i];
    v.y = vel[3 * i + 1];
    v.z = vel[3 * i + 2];
  }
  p.vel[buf][i] = v;
  p.force[i] = make_float4(0.f, 0.f, 0.f, 0.f);
}

__global__ void k_unpack(DevP p, float* __restrict__ pos, float* __restrict__ vel, float* __restrict__ force,
                         float* __restrict__ rho) {
  unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.N) return;
  const unsigned cur = p.ctl->cur;
  float4 x = p.pos[cur][i], v = p.vel[cur][i], f = p.force[i];
  unsigned tag = f2u(x.w) & 0x7FFFFFFFu;
  if (pos) { pos[3 * tag] = x.x; pos[3 * tag + 1] = x.y; pos[3 * tag + 2] = x.z; }
  if (vel) { vel[3 * tag] = v.x; vel[3 * tag + 1] = v.y; vel[3 * tag + 2] = v.z; }
  if (force) { force[3 * tag] = f.x; force[3 * tag + 1] = f.y; force[3 * tag + 2] = f.z; }
  if (rho) rho[tag] = v.w;
}

__global__ void k_count_in_solid(DevP p, unsigned* count) {
  unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.N) return;
  float4 x = p.pos[p.ctl->cur][i];
  if (f2u(x.w) >> 31) return;
  int ix = min((int)(x.x * p.inv_voxel), p.mx - 1), iy = min((int)(x.y * p.inv_voxel), p.my - 1),
      iz = min((int)(x.z * p.inv_voxel), p.mz - 1);
  if (p.mask[((size_t)iz * p.my + iy) * p.mx + ix]) atomicAdd(count, 1u);
}

// ----------------------------------------------------------------------------------------------------------------
// a7 + a8 + a4: velocity-Verlet kicks, drift, wrap, bounce-back, displacement trigger (Algorithm 1 lines 1 and 7).
// do_B: second half kick of the step just finished; do_A: first half kick + drift of the next step.
// ----------------------------------------------------------------------------------------------------------------
template <bool HAS_MASK>
__global__ void __launch_bounds__(TPB) k_integrate(const DevP p, int do_B, int do_A) {
  const unsigned cur = p.ctl->cur;
  const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
  float d2 = 0.0f;
  unsigned bounced = 0, bad = 0;
  if (i < p.N) {
    float4 x = p.pos[cur][i];
    if (!(f2u(x.w) >> 31)) {  // fluid; frozen particles are never integrated (R8)
      float4 v = p.vel[cur][i];
      const float4 f = p.force[i];
      if (do_B) {
        v.x += p.hdt_m * f.x;
        v.y += p.hdt_m * f.y;
        v.z += p.hdt_m * f.z;
      }
      if (do_A) {
        v.x += p.hdt_m * f.x;
        v.y += p.hdt_m * f.y;
        v.z += p.hdt_m * f.z;
        float nx = wrap1(x.x + p.dt * v.x, p.Lx);
        float ny = wrap1(x.y + p.dt * v.y, p.Ly);
        float nz = wrap1(x.z + p.dt * v.z, p.Lz);
        bool solid = false;
        if (HAS_MASK) {
          int ix = min((int)(nx * p.inv_voxel), p.mx - 1), iy = min((int)(ny * p.inv_voxel), p.my - 1),
              iz = min((int)(nz * p.inv_voxel), p.mz - 1);
          if (!(nx == nx && ny == ny && nz == nz)) ix = iy = iz = 0;
          solid = p.mask[((size_t)iz * p.my + iy) * p.mx + ix] != 0;
        }
        if (solid) {  // bounce-back (R7): position kept, velocity reversed
          v.x = -v.x;
          v.y = -v.y;
          v.z = -v.z;
          bounced = 1;
        } else {
          x.x = nx;
          x.y = ny;
          x.z = nz;
        }
        const float4 xb = p.xbuild[i];
        float dx = minimg(x.x - xb.x, p.Lx), dy = minimg(x.y - xb.y, p.Ly), dz = minimg(x.z - xb.z, p.Lz);
        d2 = dx * dx + dy * dy + dz * dz;
        if (!(d2 < 1e30f)) {
          bad = 1;
          d2 = 0.0f;
        }
        p.pos[cur][i] = x;
      }
      p.vel[cur][i] = v;
    }
  }
  if (!do_A) return;
  // block reduction of the trigger quantities
  unsigned m = f2u(d2);  // non-negative floats order like their bit patterns
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
  unsigned nb = __reduce_add_sync(0xffffffffu, bounced);
  unsigned nbad = __reduce_add_sync(0xffffffffu, bad);
  __shared__ unsigned s_m[TPB / 32], s_b[TPB / 32], s_n[TPB / 32];
  __shared__ bool s_last;
  const int w = threadIdx.x >> 5;
  if ((threadIdx.x & 31) == 0) {
    s_m[w] = m;
    s_b[w] = nb;
    s_n[w] = nbad;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned mm = 0, bb = 0, nn = 0;
    for (int k = 0; k < TPB / 32; ++k) {
      mm = max(mm, s_m[k]);
      bb += s_b[k];
      nn += s_n[k];
    }
    Ctl* c = p.ctl;
    if (mm) atomicMax(&c->maxdisp2, mm);
    if (bb) atomicAdd(&c->bounces, (unsigned long long)bb);
    if (nn) {
      atomicAdd(&c->nan_events, (unsigned long long)nn);
      atomicOr(&c->err, ERR_NAN);
    }
    __threadfence();
    unsigned t = atomicAdd(&c->ticket, 1u);
    s_last = (t == gridDim.x - 1);
    if (s_last) {  // every block has published its maximum: decide the rebuild for this step
      __threadfence();
      unsigned md = atomicOr(&c->maxdisp2, 0u);
      unsigned rb = u2f(md) > p.thr2 ? 1u : 0u;
      c->rebuild = rb;
      if (rb) {
        c->cur = cur ^ 1u;
        c->maxdisp2 = 0u;
        c->rebuilds += 1ull;
      }
      c->step += 1u;
      c->steps += 1ull;
      c->ticket = 0u;
    }
  }
}

// ----------------------------------------------------------------------------------------------------------------
// a1 + a2: counting sort of particles into Morton-ordered cells (every kernel of the chain is predicated on
// ctl->rebuild; src = cur ^ 1 holds the old order, dst = cur receives the new one).
// ----------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(TPB) k_cell_count(const DevP p) {
  if (!p.ctl->rebuild) return;
  const unsigned src = p.ctl->cur ^ 1u;
  unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.N) return;
  float4 x = p.pos[src][i];
  int cx = cell_coord(x.x, p.icx, p.ncx), cy = cell_coord(x.y, p.icy, p.ncy), cz = cell_coord(x.z, p.icz, p.ncz);
  unsigned c = p.cell_rank[((unsigned)cz * p.ncy + cy) * p.ncx + cx];
  p.pcell[i] = c;
  atomicAdd(&p.cell_count[c], 1u);
}

// exclusive scan of cell_count[0..ncell) into cell_start, three kernels
__global__ void __launch_bounds__(SCAN_TPB) k_scan_local(const DevP p) {
  if (!p.ctl->rebuild) return;
  const unsigned base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
  unsigned v[SCAN_ITEMS];
  unsigned sum = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) {
    unsigned idx = base + k;
    v[k] = idx < p.ncell ? p.cell_count[idx] : 0u;
    sum += v[k];
  }
  // block exclusive scan of the per-thread sums
  unsigned incl = sum;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    unsigned t = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += t;
  }
  __shared__ unsigned s_w[SCAN_TPB / 32];
  if (lane == 31) s_w[w] = incl;
  __syncthreads();
  unsigned woff = 0;
  for (int k = 0; k < w; ++k) woff += s_w[k];
  unsigned run = woff + incl - sum;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) {
    unsigned idx = base + k;
    if (idx < p.ncell) p.cell_start[idx] = run;
    run += v[k];
  }
  if (threadIdx.x == SCAN_TPB - 1) p.scan_bsum[blockIdx.x] = run;
}

__global__ void __launch_bounds__(1024) k_scan_bsum(const DevP p, unsigned nb) {
  if (!p.ctl->rebuild) return;
  __shared__ unsigned s_w[32];
  __shared__ unsigned s_carry;
  if (threadIdx.x == 0) s_carry = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (unsigned b0 = 0; b0 < nb; b0 += 1024) {
    unsigned idx = b0 + threadIdx.x;
    unsigned v = idx < nb ? p.scan_bsum[idx] : 0u;
    unsigned incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      unsigned t = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += t;
    }
    if (lane == 31) s_w[w] = incl;
    __syncthreads();
    unsigned woff = 0;
    for (int k = 0; k < w; ++k) woff += s_w[k];
    unsigned carry = s_carry;
    if (idx < nb) p.scan_bsum[idx] = carry + woff + incl - v;
    __syncthreads();
    if (threadIdx.x == 1023) s_carry = carry + woff + incl;
    __syncthreads();
  }
}

__global__ void __launch_bounds__(SCAN_TPB) k_scan_add(const DevP p) {
  if (!p.ctl->rebuild) return;
  const unsigned off = p.scan_bsum[blockIdx.x];
  const unsigned base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) {
    unsigned idx = base + k;
    if (idx < p.ncell) p.cell_start[idx] += off;
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) p.cell_start[p.ncell] = p.N;
}

__global__ void __launch_bounds__(TPB) k_cell_fill(const DevP p) {
  if (!p.ctl->rebuild) return;
  unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.N) return;
  unsigned c = p.pcell[i];
  unsigned slot = atomicSub(&p.cell_count[c], 1u) - 1u;  // the histogram counts back down to zero: self-cleaning
  p.order[p.cell_start[c] + slot] = i;
}

// Final position inside the cell = rank of the particle's tag among the cell's particles: the sorted order is a pure
// function of the positions (deterministic, independent of the atomics' arrival order).
__global__ void __launch_bounds__(TPB) k_permute(const DevP p) {
  if (!p.ctl->rebuild) return;
  const unsigned cur = p.ctl->cur, src = cur ^ 1u;
  unsigned s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= p.N) return;
  const unsigned i = p.order[s];
  const unsigned c = p.pcell[i];
  const unsigned cs = p.cell_start[c], ce = p.cell_start[c + 1];
  const float4 x = p.pos[src][i];
  const unsigned tag = f2u(x.w) & 0x7FFFFFFFu;
  unsigned rank = 0;
  for (unsigned t = cs; t < ce; ++t) {
    unsigned ot = f2u(p.pos[src][p.order[t]].w) & 0x7FFFFFFFu;
    rank += (ot < tag) ? 1u : 0u;
  }
  const unsigned dst = cs + rank;
  p.pos[cur][dst] = x;
  p.vel[cur][dst] = p.vel[src][i];
  p.xbuild[dst] = x;
}

// ----------------------------------------------------------------------------------------------------------------
// a3: Verlet list (full list; near part r < rnear = rd + skin first, far part rnear <= r < rc + skin)
// ----------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(TPB) k_build_list(const DevP p) {
  if (!p.ctl->rebuild) return;
  const unsigned cur = p.ctl->cur;
  unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
  unsigned nn = 0, nf = 0;
  bool over = false;
  if (i < p.N) {
    const float4 xi = p.pos[cur][i];
    const int cx = cell_coord(xi.x, p.icx, p.ncx), cy = cell_coord(xi.y, p.icy, p.ncy),
              cz = cell_coord(xi.z, p.icz, p.ncz);
    for (int dz = -1; dz <= 1; ++dz) {
      int oz = cz + dz;
      float sz = xi.z;
      if (oz < 0) { oz += p.ncz; sz += p.Lz; }
      else if (oz >= p.ncz) { oz -= p.ncz; sz -= p.Lz; }
      for (int dy = -1; dy <= 1; ++dy) {
        int oy = cy + dy;
        float sy = xi.y;
        if (oy < 0) { oy += p.ncy; sy += p.Ly; }
        else if (oy >= p.ncy) { oy -= p.ncy; sy -= p.Ly; }
        for (int dx = -1; dx <= 1; ++dx) {
          int ox = cx + dx;
          float sx = xi.x;
          if (ox < 0) { ox += p.ncx; sx += p.Lx; }
          else if (ox >= p.ncx) { ox -= p.ncx; sx -= p.Lx; }
          const unsigned c = p.cell_rank[((unsigned)oz * p.ncy + oy) * p.ncx + ox];
          const unsigned js = p.cell_start[c], je = p.cell_start[c + 1];
          for (unsigned j = js; j < je; ++j) {
            const float4 xj = p.pos[cur][j];
            const float ddx = sx - xj.x, ddy = sy - xj.y, ddz = sz - xj.z;
            const float r2 = ddx * ddx + ddy * ddy + ddz * ddz;
            if (r2 < p.rlist2 && j != i) {
              if (r2 < p.rnear2) {
                if (nn < p.cap_near) p.nbr_near[(size_t)nn * p.N + i] = j;
                else over = true;
                ++nn;
              } else {
                if (nf < p.cap_far) p.nbr_far[(size_t)nf * p.N + i] = j;
                else over = true;
                ++nf;
              }
            }
          }
        }
      }
    }
    p.nnbr[i] = min(nn, p.cap_near) | (min(nf, p.cap_far) << 16);
  }
  // statistics + overflow flag
  unsigned tot = nn + nf;
  unsigned wmax = __reduce_max_sync(0xffffffffu, tot);
  unsigned wsum = __reduce_add_sync(0xffffffffu, tot);
  unsigned wnear = __reduce_add_sync(0xffffffffu, nn);
  unsigned wover = __any_sync(0xffffffffu, over);
  if ((threadIdx.x & 31) == 0) {
    Ctl* c = p.ctl;
    atomicMax(&c->max_nbr, wmax);
    atomicAdd(&c->sum_nbr, (unsigned long long)wsum);
    atomicAdd(&c->sum_near, (unsigned long long)wnear);
    if (wover) {
      atomicOr(&c->err, ERR_OVERFLOW);
      atomicAdd(&c->overflow, 1ull);
    }
  }
}

__global__ void k_reset_list_stats(const DevP p) {
  if (!p.ctl->rebuild) return;
  p.ctl->max_nbr = 0;
  p.ctl->sum_nbr = 0;
  p.ctl->sum_near = 0;
}

// ----------------------------------------------------------------------------------------------------------------
// a5: density pass   rho_i = sum_{j != i, r < rd} 15 / (2 pi rd^3) (1 - r / rd)^2
// ----------------------------------------------------------------------------------------------------------------
template <bool PERIODIC>
__device__ __forceinline__ float density_loop(const DevP& p, const float4* __restrict__ pos, const float4 xi,
                                              unsigned i, unsigned nn) {
  float rho = 0.0f;
  const unsigned* __restrict__ lst = p.nbr_near + i;
#pragma unroll 4
  for (unsigned k = 0; k < nn; ++k) {
    const unsigned j = lst[(size_t)k * p.N];
    const float4 xj = __ldg(&pos[j]);
    float dx = xi.x - xj.x, dy = xi.y - xj.y, dz = xi.z - xj.z;
    if (PERIODIC) {
      dx = minimg(dx, p.Lx);
      dy = minimg(dy, p.Ly);
      dz = minimg(dz, p.Lz);
    }
    const float r2 = dx * dx + dy * dy + dz * dz;
    if (r2 < p.rd2) {
      const float r = r2 * rsqrtf(fmaxf(r2, 1e-30f));
      const float w = 1.0f - r * p.inv_rd;
      rho += w * w;
    }
  }
  return rho * p.Krho;
}

__device__ __forceinline__ bool is_interior(const DevP& p, const float4 x) {
  return x.x >= p.margin && x.x <= p.Lx - p.margin && x.y >= p.margin && x.y <= p.Ly - p.margin && x.z >= p.margin &&
         x.z <= p.Lz - p.margin;
}

__global__ void __launch_bounds__(TPB) k_density(const DevP p) {
  const unsigned cur = p.ctl->cur;
  unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.N) return;
  const float4* __restrict__ pos = p.pos[cur];
  const float4 xi = pos[i];
  const unsigned nn = p.nnbr[i] & 0xFFFFu;
  float rho;
  if (is_interior(p, xi)) rho = density_loop<false>(p, pos, xi, i, nn);
  else rho = density_loop<true>(p, pos, xi, i, nn);
  p.vel[cur][i].w = rho;
}

// ----------------------------------------------------------------------------------------------------------------
// a6: pair-force pass (Eq. (1); L186 body force)
//   F_ij = [A wC + B (rho_i + rho_j) wd - gamma wC^2 (e.v_ij) + sigma wC xi_ij / sqrt(dt)] e_ij ,  s = 1
// Full list: every pair is evaluated from both ends; the symmetric hash makes F_ij = -F_ji bitwise.
// ----------------------------------------------------------------------------------------------------------------
struct ForceAcc {
  float x, y, z;
};

template <bool PERIODIC, bool FAR>
__device__ __forceinline__ void force_loop(const DevP& p, const float4* __restrict__ pos,
                                           const float4* __restrict__ vel, const float4 xi, const float4 vi,
                                           const unsigned tagi, const unsigned walli, const HashKeys& K, unsigned i,
                                           unsigned cnt, ForceAcc& acc) {
  const unsigned* __restrict__ lst = (FAR ? p.nbr_far : p.nbr_near) + i;
#pragma unroll 2
  for (unsigned k = 0; k < cnt; ++k) {
    const unsigned j = lst[(size_t)k * p.N];
    const float4 xj = __ldg(&pos[j]);
    float dx = xi.x - xj.x, dy = xi.y - xj.y, dz = xi.z - xj.z;
    if (PERIODIC) {
      dx = minimg(dx, p.Lx);
      dy = minimg(dy, p.Ly);
      dz = minimg(dz, p.Lz);
    }
    const float r2 = dx * dx + dy * dy + dz * dz;
    const unsigned wj = f2u(xj.w);
    if (r2 < p.rc2 && r2 > 1e-12f && !(walli & (wj >> 31))) {
      const float4 vj = __ldg(&vel[j]);
      const float rinv = rsqrtf(r2);
      const float r = r2 * rinv;
      const float w = 1.0f - r * p.inv_rc;
      float F = p.A * w;
      if (!FAR) {  // pairs of the far part have r >= rd for the whole life of the list
        const float wd = fmaxf(0.0f, 1.0f - r * p.inv_rd);
        F += p.B * (vi.w + vj.w) * wd;
      }
      const float ev = (dx * (vi.x - vj.x) + dy * (vi.y - vj.y) + dz * (vi.z - vj.z)) * rinv;
      F -= p.gamma * w * w * ev;
      const unsigned h = pair_hash(tagi, wj & 0x7FFFFFFFu, K);
      const float xi_s = (float)((int)(h >> 8) - (1 << 23));  // exact
      F += p.sig_c * w * xi_s;
      const float Fr = F * rinv;
      acc.x += Fr * dx;
      acc.y += Fr * dy;
      acc.z += Fr * dz;
    }
  }
}

template <bool ALL>  // ALL: also evaluate the (never used) forces on frozen particles, for parity checks
__global__ void __launch_bounds__(TPB) k_force(const DevP p) {
  const unsigned cur = p.ctl->cur;
  unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.N) return;
  const float4* __restrict__ pos = p.pos[cur];
  const float4* __restrict__ vel = p.vel[cur];
  const float4 xi = pos[i];
  const unsigned wi = f2u(xi.w);
  const unsigned walli = wi >> 31;
  if (!ALL && walli) return;
  const float4 vi = vel[i];
  const HashKeys K = make_keys(p.ctl->step, p.seed);
  const unsigned cnt = p.nnbr[i];
  ForceAcc acc = {0.f, 0.f, 0.f};
  if (is_interior(p, xi)) {
    force_loop<false, false>(p, pos, vel, xi, vi, wi & 0x7FFFFFFFu, walli, K, i, cnt & 0xFFFFu, acc);
    force_loop<false, true>(p, pos, vel, xi, vi, wi & 0x7FFFFFFFu, walli, K, i, cnt >> 16, acc);
  } else {
    force_loop<true, false>(p, pos, vel, xi, vi, wi & 0x7FFFFFFFu, walli, K, i, cnt & 0xFFFFu, acc);
    force_loop<true, true>(p, pos, vel, xi, vi, wi & 0x7FFFFFFFu, walli, K, i, cnt >> 16, acc);
  }
  if (!walli) {
    acc.x += p.fgx;
    acc.y += p.fgy;
    acc.z += p.fgz;
  }
  p.force[i] = make_float4(acc.x, acc.y, acc.z, 0.0f);
}

// ----------------------------------------------------------------------------------------------------------------
// parity exports
// ----------------------------------------------------------------------------------------------------------------
__global__ void k_pairs(const DevP p, float rcut2, uint2* out, unsigned long long cap, unsigned long long* count) {
  const unsigned cur = p.ctl->cur;
  unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.N) return;
  const float4* __restrict__ pos = p.pos[cur];
  const float4 xi = pos[i];
  const unsigned tagi = f2u(xi.w) & 0x7FFFFFFFu;
  const unsigned cnt = p.nnbr[i];
  for (int part = 0; part < 2; ++part) {
    const unsigned n = part ? (cnt >> 16) : (cnt & 0xFFFFu);
    const unsigned* lst = (part ? p.nbr_far : p.nbr_near) + i;
    for (unsigned k = 0; k < n; ++k) {
      const unsigned j = lst[(size_t)k * p.N];
      const float4 xj = pos[j];
      const unsigned tagj = f2u(xj.w) & 0x7FFFFFFFu;
      if (tagi >= tagj) continue;
      float dx = minimg(xi.x - xj.x, p.Lx), dy = minimg(xi.y - xj.y, p.Ly), dz = minimg(xi.z - xj.z, p.Lz);
      const float r2 = dx * dx + dy * dy + dz * dz;
      if (r2 < rcut2) {
        unsigned long long s = atomicAdd(count, 1ull);
        if (s < cap) out[s] = make_uint2(tagi, tagj);
      }
    }
  }
}

__global__ void k_rng_fill(unsigned long long n, const uint2* __restrict__ pairs, unsigned step, unsigned seed,
                           unsigned* __restrict__ out) {
  unsigned long long q = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= n) return;
  const HashKeys K = make_keys(step, seed);
  out[q] = pair_hash(pairs[q].x, pairs[q].y, K);
}

// ----------------------------------------------------------------------------------------------------------------
// host side
// ----------------------------------------------------------------------------------------------------------------
inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

struct Layout {
  size_t pos[2], vel[2], force, xbuild, cell_rank, cell_count, cell_start, scan_bsum, pcell, order, nbr_near, nbr_far,
      nnbr, mask, ctl, stage, total;
  unsigned ncx, ncy, ncz, ncell, cap_near, cap_far, scan_blocks;
  float rlist, rnear;
};

bool make_layout(const mdpd_params& p, uint64_t n, int has_mask, const uint32_t* md, Layout& L, std::string* why) {
  auto fail = [&](const char* m) {
    if (why) *why = m;
    return false;
  };
  if (!(p.rc > 0) || !(p.rd > 0) || !(p.rd <= p.rc)) return fail("need 0 < rd <= rc");
  if (!(p.skin >= 0)) return fail("skin must be >= 0");
  if (!(p.dt > 0) || !(p.mass > 0)) return fail("dt and mass must be > 0");
  if (p.s != 1.0f) return fail("only s = 1 is implemented (DESIGN.md R15)");
  if (p.reorder_every > 1) return fail("only reorder_every = 0/1 is implemented (DESIGN.md R16)");
  if (n >= (1ull << 31)) return fail("n must be < 2^31");
  L.rlist = p.rc + p.skin;
  L.rnear = std::min(p.rd + p.skin, L.rlist);
  int nc[3];
  for (int d = 0; d < 3; ++d) {
    if (!(p.box[d] > 0)) return fail("box must be > 0");
    nc[d] = (int)std::floor((double)p.box[d] / (double)L.rlist);
    if (nc[d] < 3) return fail("box must hold at least 3 cells of edge rc + skin per dimension (DESIGN.md R4)");
    if (nc[d] > 1023) return fail("more than 1023 cells per dimension");
  }
  L.ncx = nc[0]; L.ncy = nc[1]; L.ncz = nc[2];
  L.ncell = (unsigned)nc[0] * nc[1] * nc[2];
  // list capacities
  const double PI = 3.14159265358979323846;
  const double vol = (double)p.box[0] * p.box[1] * p.box[2];
  const double dens = std::max(8.0, 1.3 * (double)n / vol);
  const double m_near = 4.0 / 3.0 * PI * std::pow((double)L.rnear, 3) * dens;
  const double m_far = 4.0 / 3.0 * PI * (std::pow((double)L.rlist, 3) - std::pow((double)L.rnear, 3)) * dens;
  auto cap_of = [](double m) { return (unsigned)(std::ceil((m + 6.0 * std::sqrt(m) + 8.0) / 8.0) * 8.0); };
  if (p.max_neigh == 0) {
    L.cap_near = cap_of(m_near);
    L.cap_far = m_far > 0 ? cap_of(m_far) : 8;
  } else {
    double fr = m_near / (m_near + m_far);
    L.cap_near = (unsigned)(std::ceil(p.max_neigh * fr / 8.0) * 8.0);
    L.cap_far = (unsigned)(std::ceil(p.max_neigh * (1.0 - fr) / 8.0) * 8.0) + 8;
  }
  if (L.cap_near > 65535 || L.cap_far > 65535) return fail("max_neigh too large (each part must be < 65536)");
  L.scan_blocks = (L.ncell + SCAN_TILE - 1) / SCAN_TILE;
  const size_t N = (size_t)std::max<uint64_t>(n, 1);
  size_t off = 0;
  auto take = [&](size_t bytes) {
    size_t o = off;
    off += align_up(bytes);
    return o;
  };
  L.ctl = take(sizeof(Ctl));
  L.pos[0] = take(N * 16); L.pos[1] = take(N * 16);
  L.vel[0] = take(N * 16); L.vel[1] = take(N * 16);
  L.force = take(N * 16);
  L.xbuild = take(N * 16);
  L.cell_rank = take((size_t)L.ncell * 4);
  L.cell_count = take((size_t)L.ncell * 4);
  L.cell_start = take(((size_t)L.ncell + 1) * 4);
  L.scan_bsum = take((size_t)L.scan_blocks * 4 + 4);
  L.pcell = take(N * 4);
  L.order = take(N * 4);
  L.nbr_near = take(N * 4 * L.cap_near);
  L.nbr_far = take(N * 4 * L.cap_far);
  L.nnbr = take(N * 4);
  L.stage = take(N * 40 + 64);  // load/unload staging: pos, vel, force [n][3] + rho [n] (+ type at load)
  size_t mbytes = 0;
  if (has_mask) {
    if (!md || !md[0] || !md[1] || !md[2]) return fail("mask dims missing");
    mbytes = (size_t)md[0] * md[1] * md[2];
  }
  L.mask = take(std::max<size_t>(mbytes, 16));
  L.total = off;
  return true;
}

}  // namespace

struct mdpd_ctx {
  int device = 0;
  cudaStream_t stream = nullptr;
  mdpd_params prm{};
  bool have_params = false;
  bool loaded = false;
  uint64_t n = 0;
  Layout L{};
  DevP d{};
  char* ws = nullptr;
  size_t ws_bytes = 0;
  bool ws_owned = false;
  size_t mask_cap = 0;  // bytes reserved for the mask in the workspace
  bool has_mask = false;
  uint64_t launches = 0;
  uint64_t host_step = 0;
  std::string err;
  Ctl* h_ctl = nullptr;  // pinned
  // per-kernel CUDA-event timing (mdpd_profile_begin / _end)
  bool prof_on = false;
  struct ProfRec { int slot; cudaEvent_t e0, e1; };
  std::vector<ProfRec> prof_recs;
  std::vector<cudaEvent_t> prof_pool;
};

namespace {

int set_err(mdpd_ctx* h, int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  if (h) h->err = buf;
  return code;
}

#define CU_TRY(h, call)                                                                             \
  do {                                                                                              \
    cudaError_t e__ = (call);                                                                       \
    if (e__ != cudaSuccess)                                                                         \
      return set_err(h, MDPD_ECUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e__), __FILE__, __LINE__); \
  } while (0)

inline unsigned nblk(uint64_t n, int tpb) { return (unsigned)((n + tpb - 1) / tpb); }

enum ProfSlot { PS_INTEGRATE = 0, PS_CELL_COUNT, PS_SCAN, PS_CELL_FILL, PS_PERMUTE, PS_BUILD_LIST, PS_DENSITY, PS_FORCE,
                PS_OTHER, PS_COUNT };
const char* const kProfNames[PS_COUNT] = {"k_integrate", "k_cell_count", "k_scan", "k_cell_fill", "k_permute",
                                          "k_build_list", "k_density", "k_force", "other"};

cudaEvent_t prof_event(mdpd_ctx* h) {
  cudaEvent_t e = nullptr;
  if (!h->prof_pool.empty()) {
    e = h->prof_pool.back();
    h->prof_pool.pop_back();
  } else {
    cudaEventCreate(&e);
  }
  return e;
}

// Every kernel launch of the step path goes through here: counts the launch and, while profiling is on, brackets it
// with CUDA events on the handle's stream.
#define LAUNCH(h, slot, ...)                                     \
  do {                                                           \
    mdpd_ctx::ProfRec r__{slot, nullptr, nullptr};               \
    if ((h)->prof_on) {                                          \
      r__.e0 = prof_event(h);                                    \
      r__.e1 = prof_event(h);                                    \
      cudaEventRecord(r__.e0, (h)->stream);                      \
    }                                                            \
    __VA_ARGS__;                                                 \
    if ((h)->prof_on) {                                          \
      cudaEventRecord(r__.e1, (h)->stream);                      \
      (h)->prof_recs.push_back(r__);                             \
    }                                                            \
    (h)->launches += 1;                                          \
  } while (0)

void fill_devp(mdpd_ctx* h) {
  const mdpd_params& p = h->prm;
  const Layout& L = h->L;
  DevP& d = h->d;
  char* w = h->ws;
  d.pos[0] = (float4*)(w + L.pos[0]); d.pos[1] = (float4*)(w + L.pos[1]);
  d.vel[0] = (float4*)(w + L.vel[0]); d.vel[1] = (float4*)(w + L.vel[1]);
  d.force = (float4*)(w + L.force);
  d.xbuild = (float4*)(w + L.xbuild);
  d.cell_rank = (unsigned*)(w + L.cell_rank);
  d.cell_count = (unsigned*)(w + L.cell_count);
  d.cell_start = (unsigned*)(w + L.cell_start);
  d.scan_bsum = (unsigned*)(w + L.scan_bsum);
  d.pcell = (unsigned*)(w + L.pcell);
  d.order = (unsigned*)(w + L.order);
  d.nbr_near = (unsigned*)(w + L.nbr_near);
  d.nbr_far = (unsigned*)(w + L.nbr_far);
  d.nnbr = (unsigned*)(w + L.nnbr);
  d.mask = (const unsigned char*)(w + L.mask);
  d.ctl = (Ctl*)(w + L.ctl);
  d.N = (unsigned)h->n;
  d.ncell = L.ncell;
  d.cap_near = L.cap_near;
  d.cap_far = L.cap_far;
  d.ncx = L.ncx; d.ncy = L.ncy; d.ncz = L.ncz;
  d.Lx = p.box[0]; d.Ly = p.box[1]; d.Lz = p.box[2];
  d.icx = (float)((double)L.ncx / (double)p.box[0]);
  d.icy = (float)((double)L.ncy / (double)p.box[1]);
  d.icz = (float)((double)L.ncz / (double)p.box[2]);
  d.rlist2 = L.rlist * L.rlist;
  d.rnear2 = L.rnear * L.rnear;
  d.margin = L.rlist + p.skin + 1e-3f;
}

void fill_physics(mdpd_ctx* h) {
  const mdpd_params& p = h->prm;
  DevP& d = h->d;
  d.rc2 = p.rc * p.rc;
  d.rd2 = p.rd * p.rd;
  d.inv_rc = 1.0f / p.rc;
  d.inv_rd = 1.0f / p.rd;
  d.Krho = (float)(15.0 / (2.0 * 3.14159265358979323846 * std::pow((double)p.rd, 3)));
  d.A = p.A; d.B = p.B; d.gamma = p.gamma;
  d.sig_c = (float)((double)p.sigma * std::sqrt(3.0) * std::ldexp(1.0, -23) / std::sqrt((double)p.dt));
  d.dt = p.dt;
  d.hdt_m = (float)(0.5 * (double)p.dt / (double)p.mass);
  d.fgx = p.mass * p.g[0]; d.fgy = p.mass * p.g[1]; d.fgz = p.mass * p.g[2];
  d.thr2 = 0.25f * p.skin * p.skin;
  d.seed = p.seed;
}

// Morton (Z-curve) rank of every cell: walk the codes of the bounding power-of-two cube in increasing order.
void build_morton_ranks(const Layout& L, std::vector<unsigned>& rank) {
  rank.assign(L.ncell, 0u);
  unsigned mx = std::max(L.ncx, std::max(L.ncy, L.ncz));
  int bits = 0;
  while ((1u << bits) < mx) ++bits;
  auto compact = [](unsigned long long v) {  // every third bit
    unsigned r = 0;
    for (int b = 0; b < 10; ++b) r |= (unsigned)((v >> (3 * b)) & 1ull) << b;
    return r;
  };
  unsigned next = 0;
  const unsigned long long ncodes = 1ull << (3 * bits);
  for (unsigned long long code = 0; code < ncodes; ++code) {
    unsigned cx = compact(code), cy = compact(code >> 1), cz = compact(code >> 2);
    if (cx < L.ncx && cy < L.ncy && cz < L.ncz) rank[((size_t)cz * L.ncy + cy) * L.ncx + cx] = next++;
  }
}

int launch_rebuild_chain(mdpd_ctx* h) {
  const DevP& d = h->d;
  const unsigned nb = nblk(h->n, TPB);
  cudaStream_t s = h->stream;
  LAUNCH(h, PS_OTHER, (k_reset_list_stats<<<1, 1, 0, s>>>(d)));
  LAUNCH(h, PS_CELL_COUNT, (k_cell_count<<<nb, TPB, 0, s>>>(d)));
  LAUNCH(h, PS_SCAN, (k_scan_local<<<h->L.scan_blocks, SCAN_TPB, 0, s>>>(d)));
  LAUNCH(h, PS_SCAN, (k_scan_bsum<<<1, 1024, 0, s>>>(d, h->L.scan_blocks)));
  LAUNCH(h, PS_SCAN, (k_scan_add<<<h->L.scan_blocks, SCAN_TPB, 0, s>>>(d)));
  LAUNCH(h, PS_CELL_FILL, (k_cell_fill<<<nb, TPB, 0, s>>>(d)));
  LAUNCH(h, PS_PERMUTE, (k_permute<<<nb, TPB, 0, s>>>(d)));
  LAUNCH(h, PS_BUILD_LIST, (k_build_list<<<nb, TPB, 0, s>>>(d)));
  return MDPD_OK;
}

int launch_forces(mdpd_ctx* h, bool all) {
  const DevP& d = h->d;
  const unsigned nb = nblk(h->n, TPB);
  LAUNCH(h, PS_DENSITY, (k_density<<<nb, TPB, 0, h->stream>>>(d)));
  if (all) LAUNCH(h, PS_FORCE, (k_force<true><<<nb, TPB, 0, h->stream>>>(d)));
  else LAUNCH(h, PS_FORCE, (k_force<false><<<nb, TPB, 0, h->stream>>>(d)));
  return MDPD_OK;
}

int launch_integrate(mdpd_ctx* h, int do_B, int do_A) {
  const unsigned nb = nblk(h->n, TPB);
  if (h->has_mask) LAUNCH(h, PS_INTEGRATE, (k_integrate<true><<<nb, TPB, 0, h->stream>>>(h->d, do_B, do_A)));
  else LAUNCH(h, PS_INTEGRATE, (k_integrate<false><<<nb, TPB, 0, h->stream>>>(h->d, do_B, do_A)));
  return MDPD_OK;
}

// synchronise, fetch the control block, translate latched device faults
int sync_and_check(mdpd_ctx* h) {
  CU_TRY(h, cudaMemcpyAsync(h->h_ctl, h->d.ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, h->stream));
  CU_TRY(h, cudaStreamSynchronize(h->stream));
  CU_TRY(h, cudaGetLastError());
  if (h->h_ctl->err & ERR_NAN)
    return set_err(h, MDPD_ENAN, "non-finite coordinates appeared (%llu events)", h->h_ctl->nan_events);
  if (h->h_ctl->err & ERR_OVERFLOW)
    return set_err(h, MDPD_EOVERFLOW,
                   "neighbour list capacity exceeded (near %u, far %u; longest list needed %u): raise max_neigh",
                   h->L.cap_near, h->L.cap_far, h->h_ctl->max_nbr);
  return MDPD_OK;
}

}  // namespace

// ================================================================================================================
// C-ABI
// ================================================================================================================
extern "C" {

int mdpd_create(mdpd_ctx** out, int device, void* cuda_stream) {
  if (!out) return MDPD_EINVAL;
  *out = nullptr;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0 || device < 0 || device >= ndev) {
    cudaGetLastError();
    return MDPD_ECUDA;  // no CPU fallback
  }
  if (cudaSetDevice(device) != cudaSuccess) return MDPD_ECUDA;
  mdpd_ctx* h = new (std::nothrow) mdpd_ctx();
  if (!h) return MDPD_ENOMEM;
  h->device = device;
  h->stream = (cudaStream_t)cuda_stream;
  if (cudaMallocHost((void**)&h->h_ctl, sizeof(Ctl)) != cudaSuccess) {
    delete h;
    return MDPD_ECUDA;
  }
  *out = h;
  return MDPD_OK;
}

int mdpd_destroy(mdpd_ctx* h) {
  if (!h) return MDPD_EINVAL;
  cudaSetDevice(h->device);
  cudaStreamSynchronize(h->stream);
  if (h->ws_owned && h->ws) cudaFree(h->ws);
  if (h->h_ctl) cudaFreeHost(h->h_ctl);
  for (auto& r : h->prof_recs) {
    cudaEventDestroy(r.e0);
    cudaEventDestroy(r.e1);
  }
  for (auto e : h->prof_pool) cudaEventDestroy(e);
  delete h;
  return MDPD_OK;
}

const char* mdpd_last_error(const mdpd_ctx* h) { return h ? h->err.c_str() : "null handle"; }

int mdpd_set_params(mdpd_ctx* h, const mdpd_params* p) {
  if (!h || !p) return MDPD_EINVAL;
  Layout L;
  std::string why;
  uint32_t md[3] = {1, 1, 1};
  if (!make_layout(*p, h->loaded ? h->n : 1, 0, md, L, &why)) return set_err(h, MDPD_EINVAL, "%s", why.c_str());
  if (p->kT > 0 && std::fabs(p->sigma * p->sigma - 2.0f * p->gamma * p->kT) > 1e-3f * std::max(1.0f, p->sigma * p->sigma))
    return set_err(h, MDPD_EINVAL, "sigma^2 != 2 gamma kT (PAPER.md L75)");
  if (h->loaded) {
    const mdpd_params& q = h->prm;
    if (memcmp(q.box, p->box, sizeof q.box) || q.rc != p->rc || q.rd != p->rd || q.skin != p->skin ||
        q.max_neigh != p->max_neigh || q.mass != p->mass)
      return set_err(h, MDPD_ESTATE, "box, cut-offs, skin, mass and capacities are frozen after load_particles");
    h->prm = *p;
    fill_physics(h);
    return MDPD_OK;
  }
  h->prm = *p;
  h->have_params = true;
  return MDPD_OK;
}

size_t mdpd_workspace_bytes(const mdpd_params* p, uint64_t n, int has_mask, const uint32_t mask_dims[3]) {
  if (!p) return 0;
  Layout L;
  if (!make_layout(*p, n, has_mask, mask_dims, L, nullptr)) return 0;
  return L.total;
}

int mdpd_set_workspace(mdpd_ctx* h, void* dev_ptr, size_t bytes) {
  if (!h || !dev_ptr) return MDPD_EINVAL;
  if (h->loaded) return set_err(h, MDPD_ESTATE, "set_workspace must precede load_particles");
  if (((uintptr_t)dev_ptr & 255u) != 0) return set_err(h, MDPD_EINVAL, "workspace must be 256-byte aligned");
  if (h->ws_owned && h->ws) cudaFree(h->ws);
  h->ws = (char*)dev_ptr;
  h->ws_bytes = bytes;
  h->ws_owned = false;
  return MDPD_OK;
}

int mdpd_load_particles(mdpd_ctx* h, uint64_t n, const float* pos, const float* vel, const uint8_t* type) {
  if (!h) return MDPD_EINVAL;
  if (!h->have_params) return set_err(h, MDPD_ESTATE, "set_params first");
  if (n && (!pos || !vel)) return set_err(h, MDPD_EINVAL, "pos / vel are NULL");
  CU_TRY(h, cudaSetDevice(h->device));
  std::string why;
  Layout L;
  // reserve mask space if the caller sized the workspace for one: recompute with the largest mask that fits
  uint32_t nomask[3] = {1, 1, 1};
  if (!make_layout(h->prm, n, 0, nomask, L, &why)) return set_err(h, MDPD_EINVAL, "%s", why.c_str());
  if (!h->ws) {
    h->ws_bytes = L.total + (64u << 20);  // room for a mask of up to 64 Mi voxels
    CU_TRY(h, cudaMalloc((void**)&h->ws, h->ws_bytes));
    h->ws_owned = true;
  }
  if (h->ws_bytes < L.total)
    return set_err(h, MDPD_ENOMEM, "workspace too small: %zu bytes given, %zu needed", h->ws_bytes, L.total);
  h->mask_cap = h->ws_bytes - L.mask;
  h->L = L;
  h->n = n;
  h->has_mask = false;
  h->loaded = false;
  fill_devp(h);
  fill_physics(h);
  // control block
  Ctl c0;
  memset(&c0, 0, sizeof c0);
  c0.cur = 1;      // the initial sort reads buffer 0 and writes buffer 1
  c0.rebuild = 1;
  c0.rebuilds = 1;
  CU_TRY(h, cudaMemcpyAsync(h->d.ctl, &c0, sizeof c0, cudaMemcpyHostToDevice, h->stream));
  CU_TRY(h, cudaStreamSynchronize(h->stream));  // c0 is on the stack
  h->host_step = 0;
  {  // Morton rank table
    std::vector<unsigned> rank;
    build_morton_ranks(L, rank);
    CU_TRY(h, cudaMemcpyAsync(h->d.cell_rank, rank.data(), rank.size() * 4, cudaMemcpyHostToDevice, h->stream));
    CU_TRY(h, cudaMemsetAsync(h->d.cell_count, 0, (size_t)L.ncell * 4, h->stream));
    CU_TRY(h, cudaStreamSynchronize(h->stream));
  }
  if (n) {
    char* st = h->ws + L.stage;
    float* spos = (float*)st;
    float* svel = spos + 3 * n;
    unsigned char* stype = (unsigned char*)(svel + 3 * n);
    CU_TRY(h, cudaMemcpyAsync(spos, pos, n * 12, cudaMemcpyDefault, h->stream));
    CU_TRY(h, cudaMemcpyAsync(svel, vel, n * 12, cudaMemcpyDefault, h->stream));
    if (type) CU_TRY(h, cudaMemcpyAsync(stype, type, n, cudaMemcpyDefault, h->stream));
    LAUNCH(h, PS_OTHER, (k_pack<<<nblk(n, TPB), TPB, 0, h->stream>>>(h->d, spos, svel, type ? stype : nullptr, 0u)));
    launch_rebuild_chain(h);
    launch_forces(h, true);
  }
  h->loaded = true;
  return sync_and_check(h);
}

int mdpd_load_wall_mask(mdpd_ctx* h, const uint8_t* mask, const uint32_t dims[3], float voxel) {
  if (!h) return MDPD_EINVAL;
  if (!h->loaded) return set_err(h, MDPD_ESTATE, "load_particles first");
  CU_TRY(h, cudaSetDevice(h->device));
  if (!mask) {
    h->has_mask = false;
    return MDPD_OK;
  }
  if (!dims || !(voxel > 0)) return set_err(h, MDPD_EINVAL, "dims / voxel missing");
  for (int k = 0; k < 3; ++k)
    if (std::fabs((double)dims[k] * voxel - h->prm.box[k]) > 1e-4 * h->prm.box[k])
      return set_err(h, MDPD_EINVAL, "mask dims * voxel must equal the box");
  size_t bytes = (size_t)dims[0] * dims[1] * dims[2];
  if (bytes > h->mask_cap)
    return set_err(h, MDPD_ENOMEM, "workspace has %zu bytes for the mask, %zu needed", h->mask_cap, bytes);
  CU_TRY(h, cudaMemcpyAsync((void*)h->d.mask, mask, bytes, cudaMemcpyDefault, h->stream));
  h->d.mx = dims[0]; h->d.my = dims[1]; h->d.mz = dims[2];
  h->d.inv_voxel = 1.0f / voxel;
  h->has_mask = true;
  if (h->n) {
    unsigned* cnt = (unsigned*)(h->ws + h->L.stage);
    CU_TRY(h, cudaMemsetAsync(cnt, 0, 4, h->stream));
    LAUNCH(h, PS_OTHER, (k_count_in_solid<<<nblk(h->n, TPB), TPB, 0, h->stream>>>(h->d, cnt)));
    unsigned bad = 0;
    CU_TRY(h, cudaMemcpyAsync(&bad, cnt, 4, cudaMemcpyDeviceToHost, h->stream));
    CU_TRY(h, cudaStreamSynchronize(h->stream));
    if (bad) return set_err(h, MDPD_EINSOLID, "%u fluid particles start inside solid voxels", bad);
  }
  return MDPD_OK;
}

int mdpd_step(mdpd_ctx* h, uint32_t nsteps) {
  if (!h) return MDPD_EINVAL;
  if (!h->loaded) return set_err(h, MDPD_ESTATE, "load_particles first");
  if (nsteps == 0) return MDPD_OK;
  h->host_step += nsteps;
  if (h->n == 0) return MDPD_OK;
  CU_TRY(h, cudaSetDevice(h->device));
  for (uint32_t it = 0; it < nsteps; ++it) {
    launch_integrate(h, it > 0, 1);  // [second half kick of the previous step +] half kick, drift, bounce, trigger
    launch_rebuild_chain(h);         // runs only if the trigger fired (device-side predicate)
    launch_forces(h, false);         // Algorithm 1 lines 4 and 6 at the new time level, half-step velocities
  }
  launch_integrate(h, 1, 0);  // Algorithm 1 line 7
  CU_TRY(h, cudaGetLastError());
  return MDPD_OK;
}

int mdpd_compute_forces(mdpd_ctx* h) {
  if (!h) return MDPD_EINVAL;
  if (!h->loaded) return set_err(h, MDPD_ESTATE, "load_particles first");
  if (h->n == 0) return MDPD_OK;
  CU_TRY(h, cudaSetDevice(h->device));
  launch_forces(h, true);
  return sync_and_check(h);
}

int mdpd_set_step_counter(mdpd_ctx* h, uint64_t step) {
  if (!h) return MDPD_EINVAL;
  if (!h->loaded) return set_err(h, MDPD_ESTATE, "load_particles first");
  CU_TRY(h, cudaSetDevice(h->device));
  unsigned s32 = (unsigned)step;
  CU_TRY(h, cudaMemcpyAsync(&h->d.ctl->step, &s32, 4, cudaMemcpyHostToDevice, h->stream));
  CU_TRY(h, cudaStreamSynchronize(h->stream));
  h->host_step = step;
  return MDPD_OK;
}

int mdpd_get_state(mdpd_ctx* h, float* pos, float* vel, float* force, float* rho, uint64_t* step) {
  if (!h) return MDPD_EINVAL;
  if (!h->loaded) return set_err(h, MDPD_ESTATE, "load_particles first");
  CU_TRY(h, cudaSetDevice(h->device));
  const uint64_t n = h->n;
  if (n) {
    float* spos = (float*)(h->ws + h->L.stage);
    float* svel = spos + 3 * n;
    float* sfor = svel + 3 * n;
    float* srho = sfor + 3 * n;
    LAUNCH(h, PS_OTHER, (k_unpack<<<nblk(n, TPB), TPB, 0, h->stream>>>(h->d, pos ? spos : nullptr, vel ? svel : nullptr,
                                                                       force ? sfor : nullptr, rho ? srho : nullptr)));
    if (pos) CU_TRY(h, cudaMemcpyAsync(pos, spos, n * 12, cudaMemcpyDefault, h->stream));
    if (vel) CU_TRY(h, cudaMemcpyAsync(vel, svel, n * 12, cudaMemcpyDefault, h->stream));
    if (force) CU_TRY(h, cudaMemcpyAsync(force, sfor, n * 12, cudaMemcpyDefault, h->stream));
    if (rho) CU_TRY(h, cudaMemcpyAsync(rho, srho, n * 4, cudaMemcpyDefault, h->stream));
  }
  int rc = sync_and_check(h);
  if (step) *step = h->host_step;
  return rc;
}

int mdpd_get_counters(mdpd_ctx* h, uint64_t out[8]) {
  if (!h || !out) return MDPD_EINVAL;
  if (!h->loaded) return set_err(h, MDPD_ESTATE, "load_particles first");
  CU_TRY(h, cudaSetDevice(h->device));
  int rc = sync_and_check(h);
  const Ctl* c = h->h_ctl;
  out[0] = h->host_step;
  out[1] = c->rebuilds;
  out[2] = c->bounces;
  out[3] = c->max_nbr;
  out[4] = c->sum_nbr;
  out[5] = c->sum_near;
  out[6] = c->overflow + c->nan_events;
  out[7] = h->launches;
  return rc;
}

int mdpd_get_pairs(mdpd_ctx* h, float rcut, uint64_t* count, uint32_t* pairs, uint64_t cap) {
  if (!h || !count) return MDPD_EINVAL;
  if (!h->loaded) return set_err(h, MDPD_ESTATE, "load_particles first");
  if (!(rcut > 0) || rcut > h->L.rlist) return set_err(h, MDPD_EINVAL, "rcut must be in (0, rc + skin]");
  CU_TRY(h, cudaSetDevice(h->device));
  *count = 0;
  if (h->n == 0) return MDPD_OK;
  if (!pairs) cap = 0;
  uint2* dout = nullptr;
  unsigned long long* dcnt = nullptr;
  CU_TRY(h, cudaMalloc((void**)&dcnt, 8));
  if (cap) {
    cudaError_t e = cudaMalloc((void**)&dout, cap * 8);
    if (e != cudaSuccess) {
      cudaFree(dcnt);
      return set_err(h, MDPD_ENOMEM, "cudaMalloc of the pair buffer failed");
    }
  }
  cudaMemsetAsync(dcnt, 0, 8, h->stream);
  LAUNCH(h, PS_OTHER, (k_pairs<<<nblk(h->n, TPB), TPB, 0, h->stream>>>(h->d, rcut * rcut, dout, cap, dcnt)));
  unsigned long long c = 0;
  cudaMemcpyAsync(&c, dcnt, 8, cudaMemcpyDeviceToHost, h->stream);
  cudaError_t e = cudaStreamSynchronize(h->stream);
  if (e == cudaSuccess && cap) {
    uint64_t m = std::min<uint64_t>(c, cap);
    e = cudaMemcpy(pairs, dout, m * 8, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) {
      std::vector<uint64_t> keys(m);  // (a << 32 | b): sorts by a, then b
      for (uint64_t q = 0; q < m; ++q) keys[q] = ((uint64_t)pairs[2 * q] << 32) | pairs[2 * q + 1];
      std::sort(keys.begin(), keys.end());
      for (uint64_t q = 0; q < m; ++q) {
        pairs[2 * q] = (uint32_t)(keys[q] >> 32);
        pairs[2 * q + 1] = (uint32_t)keys[q];
      }
    }
  }
  cudaFree(dcnt);
  if (dout) cudaFree(dout);
  if (e != cudaSuccess) return set_err(h, MDPD_ECUDA, "get_pairs: %s", cudaGetErrorString(e));
  *count = c;
  return MDPD_OK;
}

int mdpd_rng_fill(mdpd_ctx* h, uint64_t npairs, const uint32_t* pairs, uint32_t step, uint32_t* out) {
  if (!h) return MDPD_EINVAL;
  if (!h->have_params) return set_err(h, MDPD_ESTATE, "set_params first");
  if (npairs == 0) return MDPD_OK;
  if (!pairs || !out) return MDPD_EINVAL;
  CU_TRY(h, cudaSetDevice(h->device));
  uint2* dp = nullptr;
  unsigned* dout = nullptr;
  CU_TRY(h, cudaMalloc((void**)&dp, npairs * 8));
  cudaError_t e = cudaMalloc((void**)&dout, npairs * 4);
  if (e != cudaSuccess) {
    cudaFree(dp);
    return set_err(h, MDPD_ENOMEM, "cudaMalloc failed in rng_fill");
  }
  cudaMemcpyAsync(dp, pairs, npairs * 8, cudaMemcpyDefault, h->stream);
  LAUNCH(h, PS_OTHER, (k_rng_fill<<<nblk(npairs, 256), 256, 0, h->stream>>>(npairs, dp, step, h->prm.seed, dout)));
  cudaMemcpyAsync(out, dout, npairs * 4, cudaMemcpyDefault, h->stream);
  e = cudaStreamSynchronize(h->stream);
  cudaFree(dp);
  cudaFree(dout);
  if (e != cudaSuccess) return set_err(h, MDPD_ECUDA, "rng_fill: %s", cudaGetErrorString(e));
  return MDPD_OK;
}

int mdpd_profile_begin(mdpd_ctx* h) {
  if (!h) return MDPD_EINVAL;
  for (auto& r : h->prof_recs) {
    h->prof_pool.push_back(r.e0);
    h->prof_pool.push_back(r.e1);
  }
  h->prof_recs.clear();
  h->prof_on = true;
  return MDPD_OK;
}

int mdpd_profile_end(mdpd_ctx* h, double ms[MDPD_PROF_SLOTS], uint64_t launches[MDPD_PROF_SLOTS]) {
  if (!h || !ms || !launches) return MDPD_EINVAL;
  static_assert(PS_COUNT <= MDPD_PROF_SLOTS, "profile slots");
  h->prof_on = false;
  CU_TRY(h, cudaSetDevice(h->device));
  CU_TRY(h, cudaStreamSynchronize(h->stream));
  for (int k = 0; k < MDPD_PROF_SLOTS; ++k) {
    ms[k] = 0.0;
    launches[k] = 0;
  }
  for (auto& r : h->prof_recs) {
    float t = 0.f;
    if (cudaEventElapsedTime(&t, r.e0, r.e1) == cudaSuccess) {
      ms[r.slot] += (double)t;
      launches[r.slot] += 1;
    }
    h->prof_pool.push_back(r.e0);
    h->prof_pool.push_back(r.e1);
  }
  h->prof_recs.clear();
  return MDPD_OK;
}

const char* mdpd_profile_name(int slot) { return (slot >= 0 && slot < PS_COUNT) ? kProfNames[slot] : ""; }

}  // extern "C"
