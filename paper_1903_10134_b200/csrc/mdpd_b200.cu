// mdpd_b200.cu -- hand-written CUDA (sm_100a) for one mDPD velocity-Verlet timestep + the C-ABI of include/mdpd.h.
//
// Paper: arxiv/paper_1903_10134.  Eq. (1) and the weight functions: PAPER.md L75-81; Algorithm 1
// (x -> rho -> f -> v): PAPER.md L125-133; body force: L186; frozen walls: L162.  Readings R1..R18 and the hash
// specification: DESIGN.md sections 3 and 4.  This file shares nothing with oracle/ (the fp64 CPU oracle).
//
// Device state: pos float4 = (x, y, z, bits(tag | species << 28 | frozen << 31)), vel float4 = (vx, vy, vz, rho),
// both double-buffered for the counting sort into tiles of cells (tiles along the Z-curve, cells x-fastest inside a
// tile); force float4; xbuild float4 (positions at the last list build); Verlet list of 16-bit indices into the
// tile's staged shared-memory image, stored in 16-byte chunks of 8 entries, layout [chunk][particle]; per tile a
// staging recipe (runs of contiguous halo cells) and per particle the hand-out records of the two per-step passes.
#include "mdpd.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

namespace {

constexpr unsigned ERR_OVERFLOW = 1u;
constexpr unsigned ERR_NAN = 2u;
constexpr unsigned ERR_TILE = 4u;  // a tile + halo does not fit the shared-memory capacity
constexpr unsigned ERR_TYPE = 8u;  // a particle's species index is not below the number of species
constexpr unsigned ERR_CHECK = 16u;  // -DMDPD_CHECKS: an internal bounds check failed (reported as MDPD_ECUDA)
// Bounds checks of the kernels' own index arithmetic (every index into the staged image, the row buffers, the lists and
// the particle arrays), compiled in with -DMDPD_CHECKS (python -m paper_1903_10134_b200.build --force -DMDPD_CHECKS) and
// run over the whole GPU test suite: this pool has compute-sanitizer closed, see profiles/sanitizer_r2.md.
#ifdef MDPD_CHECKS
#define MDPD_CHECK(p, cond)                              \
  do {                                                   \
    if (!(cond)) atomicOr(&(p).ctl->err, ERR_CHECK);     \
  } while (0)
#else
#define MDPD_CHECK(p, cond) ((void)0)
#endif
// particle word (pos.w): tag (load-order index) | species << 28 | frozen << 31
constexpr unsigned TAG_BITS = 28, TAG_MASK = (1u << TAG_BITS) - 1u, MAXTYPES = 8;
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
  unsigned max_halo;  // most particles in a tile + halo at the last build
  unsigned max_own;   // most particles in a tile at the last build
  unsigned has_wall;  // some particle is frozen (set by k_pack)
  unsigned long long steps, rebuilds, bounces, sum_nbr, overflow, nan_events, sum_act, dens_passes, graph_rebuilds, pad2;
  double vir[6];             // k_force<.., VIRIAL>: sum over list entries of r_a F^C_b (xx, yy, zz, xy, xz, yz); each pair twice
};

struct TileInfo {  // one CTA of the list / density / force passes
  int c0x, c0y, c0z;   // first cell
  int ex, ey, ez;      // extent in cells (<= 4 each)
  unsigned rank0;      // sorted rank of the tile's first cell; its cells are ranks rank0 .. rank0 + ncell_own - 1
  unsigned ncell_own;  // ex * ey * ez
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
  uint4* nbr;                // [cap / 8][N] chunks of 8 16-bit staged-slot indices, padded with the sentinel slot
  unsigned short* self_loc;  // [N] staged slot of the particle itself
  unsigned* nnbr;            // [N] list length
  uint4* act;                // [cap / 8][N] this step's in-range (r < rc) subset of the list, written by the density pass
  unsigned short* nact;      // [N] its length
  const TileInfo* tiles;     // [ntiles]
  uint4* runs;               // [ntiles][run_stride] staging recipe of every tile, written by k_tile_recipe (see stage_fast)
  uint2* dinfo;              // [N] hand-out records of the density pass: own particles of every tile in order of decreasing
                             //     list length; x = index in the tile | own staged slot << 16, y = list length
  uint2* finfo;              // [N] ... of the force pass: in order of decreasing in-range count of this step (y = count,
                             //     bit 31: frozen particle whose force is not needed), written by the density pass
  const unsigned char* mask;
  Ctl* ctl;
  // sizes
  unsigned N, ncell, cap, ntiles, tile_cap, run_stride;
  unsigned nrun_max;     // run records per tile: 3 (ty + 2)(tz + 2)
  unsigned hb_off;       // recipe: offset (in uint4) of the tile's table of first staged slots of its halo cells (u16)
  unsigned cap_act;      // capacity of the per-step in-range (r < rc) lists of the list-free path
  unsigned rows_verlet, rows_direct;  // bytes per row of k_cells' per-warp row buffers (list build / list-free pass)
  float dot_margin;      // slack of the approximate (dot-product form) range test of k_cells, in units of r^2
  unsigned sms;          // multiprocessors of the device: a tile pass prefetches (L2) for the tile that starts one CTA lifetime later
  unsigned tma_staging;  // bit 0 / bit 1: the density / force pass stages its tile with bulk copies (stage_bulk), else cp.async (stage_fast)
  int ncx, ncy, ncz;
  int mx, my, mz;
  // geometry
  float Lx, Ly, Lz;
  float icx, icy, icz;  // 1 / cell edge
  float edge_x, edge_y, edge_z;
  float inv_voxel;
  float rlist2, rc2, rd2;
  // physics
  float inv_rc, inv_rd, Krho;
  float A, B, gamma, sig_c;  // sig_c = sigma * sqrt(3) * 2^-23 / sqrt(dt)
  float dt, hdt_m;           // dt, 0.5 dt / m
  float fgx, fgy, fgz;       // m g
  float s_exp;               // exponent s of wR = (1 - r/rc)^s; the kernels specialise s = 1
  unsigned ntypes;           // 0: one material (type byte != 0 <=> frozen); else the type byte is a species index
  unsigned frozen_mask;      // bit s: species s is frozen
  float2 AB[MAXTYPES * MAXTYPES];  // per-type-pair (A, B) of Eq. (1), row = species_i * MAXTYPES (Tables 1-2)
  float2 GS[MAXTYPES * MAXTYPES];  // per-type-pair (gamma, sig_c) of F^D, F^R (water 12.4 L141, other fluids 4.5 L89)
  float thr2;                // (skin / 2)^2
  unsigned seed;
};

__device__ __forceinline__ unsigned f2u(float f) { return __float_as_uint(f); }
__device__ __forceinline__ float rsqrt_fast(float x) {  // one MUFU.RSQ (2 ulp); callers keep x out of the denormals
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float sqrt_fast(float x) {  // one MUFU.SQRT; sqrt(0) = 0
  float y;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float u2f(unsigned u) { return __uint_as_float(u); }

// Shared-memory gathers of the hot loops go through 32-bit shared addresses (one LEA per neighbour and array).
__device__ __forceinline__ unsigned smem_addr(const void* ptr) { return (unsigned)__cvta_generic_to_shared(ptr); }
__device__ __forceinline__ float4 lds4(unsigned addr) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
  return v;
}
__device__ __forceinline__ void prefetch_l2(const void* ptr) { asm volatile("prefetch.global.L2 [%0];" ::"l"(ptr)); }
__device__ __forceinline__ unsigned pin(unsigned v) {  // keeps a loop-invariant value in its register (no rematerialisation)
  asm volatile("" : "+r"(v));
  return v;
}

// Positions are kept UNWRAPPED between list rebuilds (they leave [0, L) by at most skin / 2) so that a particle stays
// geometrically inside the cell it was sorted into; they are wrapped when the sort runs, for the voxel-mask lookup
// and on output (R12).
__device__ __forceinline__ float wrap1(float x, float L) {  // |x - [0,L)| << L here
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
  unsigned t = 0u, sp = 0u;  // frozen flag, species
  if (type) {
    if (p.ntypes) {
      sp = type[i];
      if (sp >= p.ntypes) {
        atomicOr(&p.ctl->err, ERR_TYPE);
        sp = 0u;
      }
      t = (p.frozen_mask >> sp) & 1u;
    } else {
      t = sp = type[i] != 0;
    }
  }
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
  if (t) atomicOr(&p.ctl->has_wall, 1u);
  p.pos[buf][i] = make_float4(x, y, z, u2f(i | (sp << TAG_BITS) | (t << 31)));
  float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
  if (!t) {
    v.x = vel[3 * i];
    v.y = vel[3 * i + 1];
    v.z = vel[3 * i + 2];
  }
  p.vel[buf][i] = v;
  p.force[i] = make_float4(0.f, 0.f, 0.f, 0.f);
}

// (re)start the control block for a fresh sort of buffer 0 into buffer 1; keeps has_wall and a bad-species fault
__global__ void k_ctl_init(DevP p) {
  Ctl* c = p.ctl;
  const unsigned hw = c->has_wall, et = c->err & ERR_TYPE;  // k_pack's findings survive the restart
  Ctl z;
  memset(&z, 0, sizeof z);
  z.err = et;
  z.cur = 1;
  z.rebuild = 1;
  z.rebuilds = 1;
  z.has_wall = hw;
  *c = z;
}

__global__ void k_unpack(DevP p, float* __restrict__ pos, float* __restrict__ vel, float* __restrict__ force,
                         float* __restrict__ rho) {
  unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.N) return;
  const unsigned cur = p.ctl->cur;
  float4 x = p.pos[cur][i], v = p.vel[cur][i], f = p.force[i];
  unsigned tag = f2u(x.w) & TAG_MASK;
  if (pos) { pos[3 * tag] = wrap1(x.x, p.Lx); pos[3 * tag + 1] = wrap1(x.y, p.Ly); pos[3 * tag + 2] = wrap1(x.z, p.Lz); }
  if (vel) { vel[3 * tag] = v.x; vel[3 * tag + 1] = v.y; vel[3 * tag + 2] = v.z; }
  if (force) { force[3 * tag] = f.x; force[3 * tag + 1] = f.y; force[3 * tag + 2] = f.z; }
  if (rho) rho[tag] = v.w;
}

__global__ void k_set_forces(DevP p, const float* __restrict__ force) {  // tag order -> sorted order
  unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.N) return;
  const unsigned tag = f2u(p.pos[p.ctl->cur][i].w) & TAG_MASK;
  p.force[i] = make_float4(force[3 * tag], force[3 * tag + 1], force[3 * tag + 2], 0.0f);
}

__global__ void k_count_in_solid(DevP p, unsigned* count) {
  unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.N) return;
  float4 x = p.pos[p.ctl->cur][i];
  if (f2u(x.w) >> 31) return;
  x.x = wrap1(x.x, p.Lx);
  x.y = wrap1(x.y, p.Ly);
  x.z = wrap1(x.z, p.Lz);
  int ix = max(min((int)(x.x * p.inv_voxel), p.mx - 1), 0), iy = max(min((int)(x.y * p.inv_voxel), p.my - 1), 0),
      iz = max(min((int)(x.z * p.inv_voxel), p.mz - 1), 0);
  if (p.mask[((size_t)iz * p.my + iy) * p.mx + ix]) atomicAdd(count, 1u);
}

// ----------------------------------------------------------------------------------------------------------------
// a7 + a8 + a4: velocity-Verlet kicks, drift, wrap, bounce-back, displacement trigger (Algorithm 1 lines 1 and 7).
// do_B: second half kick of the step just finished; do_A: first half kick + drift of the next step.
// ----------------------------------------------------------------------------------------------------------------
template <bool HAS_MASK>
__global__ void __launch_bounds__(TPB) k_integrate(const DevP p, int do_B, int do_A, cudaGraphConditionalHandle cond,
                                                   int use_cond) {
  const unsigned cur = p.ctl->cur;
  float d2max = 0.0f;
  unsigned bounced = 0, bad = 0;
  // grid-stride over the particles: a few waves of blocks, so that the same-address atomics of the trigger below are
  // a few thousand per launch, not one pair per 128 particles
  for (unsigned i = blockIdx.x * blockDim.x + threadIdx.x; i < p.N; i += gridDim.x * blockDim.x) {
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
        const float nx = x.x + p.dt * v.x, ny = x.y + p.dt * v.y, nz = x.z + p.dt * v.z;
        bool solid = false, fin = true;
        if (HAS_MASK) {
          const float wx = wrap1(nx, p.Lx), wy = wrap1(ny, p.Ly), wz = wrap1(nz, p.Lz);
          int ix = max(min((int)(wx * p.inv_voxel), p.mx - 1), 0), iy = max(min((int)(wy * p.inv_voxel), p.my - 1), 0),
              iz = max(min((int)(wz * p.inv_voxel), p.mz - 1), 0);
          // a trial position that is not finite, or that one period does not bring back into the box (a runaway
          // particle), is a fault (MDPD_ENAN), not a mask lookup
          fin = fabsf(nx - 0.5f * p.Lx) <= 1.5f * p.Lx && fabsf(ny - 0.5f * p.Ly) <= 1.5f * p.Ly && fabsf(nz - 0.5f * p.Lz) <= 1.5f * p.Lz;
          if (!fin) ix = iy = iz = 0;
          solid = p.mask[((size_t)iz * p.my + iy) * p.mx + ix] != 0;
        }
        if (solid) {  // bounce-back (R7): position kept, velocity reversed
          v.x = -v.x;
          v.y = -v.y;
          v.z = -v.z;
          bounced += 1;
        } else {
          x.x = nx;
          x.y = ny;
          x.z = nz;
        }
        const float4 xb = p.xbuild[i];
        const float dx = x.x - xb.x, dy = x.y - xb.y, dz = x.z - xb.z;  // unwrapped since the last build
        const float d2 = dx * dx + dy * dy + dz * dz;
        if (!(d2 < 1e30f) || !fin) bad += 1;
        else d2max = fmaxf(d2max, d2);
        p.pos[cur][i] = x;
      }
      p.vel[cur][i] = v;
    }
  }
  if (!do_A) return;
  // block reduction of the trigger quantities
  unsigned m = f2u(d2max);  // non-negative floats order like their bit patterns
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
      if (use_cond) {  // inside the step graph: the IF node that holds the rebuild chain runs only when the trigger fired
        cudaGraphSetConditional(cond, rb);
        if (rb) c->graph_rebuilds += 1ull;
      }
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
  for (unsigned i = blockIdx.x * blockDim.x + threadIdx.x; i < p.N; i += gridDim.x * blockDim.x) {
    float4 x = p.pos[src][i];
    x.x = wrap1(x.x, p.Lx);
    x.y = wrap1(x.y, p.Ly);
    x.z = wrap1(x.z, p.Lz);
    int cx = cell_coord(x.x, p.icx, p.ncx), cy = cell_coord(x.y, p.icy, p.ncy), cz = cell_coord(x.z, p.icz, p.ncz);
    unsigned c = p.cell_rank[((unsigned)cz * p.ncy + cy) * p.ncx + cx];
    p.pcell[i] = c;
    atomicAdd(&p.cell_count[c], 1u);
  }
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
  for (unsigned i = blockIdx.x * blockDim.x + threadIdx.x; i < p.N; i += gridDim.x * blockDim.x) {
    unsigned c = p.pcell[i];
    unsigned slot = atomicSub(&p.cell_count[c], 1u) - 1u;  // the histogram counts back down to zero: self-cleaning
    MDPD_CHECK(p, c < p.ncell && p.cell_start[c] + slot < p.N);
    p.order[p.cell_start[c] + slot] = i;
  }
}

// Final position inside the cell = rank of the particle's tag among the cell's particles: the sorted order is a pure
// function of the positions (deterministic, independent of the atomics' arrival order).
__global__ void __launch_bounds__(TPB) k_permute(const DevP p) {
  if (!p.ctl->rebuild) return;
  const unsigned cur = p.ctl->cur, src = cur ^ 1u;
  for (unsigned s = blockIdx.x * blockDim.x + threadIdx.x; s < p.N; s += gridDim.x * blockDim.x) {
  const unsigned i = p.order[s];
  const unsigned c = p.pcell[i];
  const unsigned cs = p.cell_start[c], ce = p.cell_start[c + 1];
  float4 x = p.pos[src][i];
  x.x = wrap1(x.x, p.Lx);
  x.y = wrap1(x.y, p.Ly);
  x.z = wrap1(x.z, p.Lz);
  const unsigned tag = f2u(x.w) & TAG_MASK;
  unsigned rank = 0;
  for (unsigned t = cs; t < ce; ++t) {
    unsigned ot = f2u(p.pos[src][p.order[t]].w) & TAG_MASK;
    rank += (ot < tag) ? 1u : 0u;
  }
  const unsigned dst = cs + rank;
  MDPD_CHECK(p, dst < p.N && i < p.N && ce <= p.N && c < p.ncell);
  p.pos[cur][dst] = x;
  p.vel[cur][dst] = p.vel[src][i];
  p.xbuild[dst] = x;
  }
}

// ----------------------------------------------------------------------------------------------------------------
// Tile staging.  A CTA owns one tile of up to 4 x 4 x 4 cells.  The tile and its one-cell halo
// (<= 6 x 6 x 6 = 216 cells) are copied once into shared memory, cell by cell in halo order (x fastest), in
// TILE-RELATIVE coordinates with the periodic shift folded in: no minimum-image arithmetic in any inner loop, and
// pair separations are formed from small numbers (|x| < 8) whatever the box size.  The Verlet list stores 16-bit
// indices into this staged array, so every neighbour access of the hot loops is a shared-memory load.
// ----------------------------------------------------------------------------------------------------------------
#ifndef MINB
#define MINB 2   // resident CTAs per SM the force pass is compiled for
#endif
#ifndef DENS_TPB
#define DENS_TPB 384  // most threads per CTA of the density pass
#endif
#ifndef DENS_TPB2
#define DENS_TPB2 416  // ... of its instantiation for fuller tiles
#endif
#ifndef DENS_MINB
#define DENS_MINB 3
#endif
#ifndef TILE_TPB
#define TILE_TPB 512  // most threads per CTA of the density / force passes (8 warps; long and short groups paired: two rounds on a full tile)
#endif
constexpr int HMAX = 216;                      // halo cells of the largest tile
constexpr int HTAB = 224;                      // table size (HMAX + 1 rounded up)
static_assert(HMAX + 1 <= HTAB, "halo table");
constexpr unsigned LCAP = 128;                 // per-particle list capacity

struct TileSmem {
  float4* spos;      // [cap + 1] (x_rel, y_rel, z_rel, particle word); slot cap = the far-away sentinel
  float4* svel;      // [cap + 1] (vx, vy, vz, rho)            (force pass only)
  float4* hshift;    // [HTAB] (sx, sy, sz, bits(delta)) of halo cell h: x_rel = x + s, global index = staged slot + delta
  unsigned* hbase;   // [HTAB] first staged slot of halo cell h; hbase[nh] = number of staged particles
  unsigned short* queue;  // scratch behind the tables (list build: per-warp rows)
};

constexpr size_t TILE_SLOT_BYTES = 32;  // pos + vel: shared-memory bytes per staged slot of the force pass

// queue_entries: 16-bit scratch entries behind the tables (list build: rows per warp)
__host__ __device__ inline size_t tile_smem_bytes(unsigned cap, bool with_vel, size_t queue_entries) {
  return (size_t)(cap + 1) * 16 * (with_vel ? 2 : 1) + HTAB * 16 + HTAB * 4 + queue_entries * 2;  // + sentinel slot
}

__device__ __forceinline__ TileSmem carve_smem(unsigned char* raw, unsigned cap, bool with_vel) {
  TileSmem s;
  s.spos = (float4*)raw;
  raw += (size_t)(cap + 1) * 16;
  s.svel = (float4*)raw;
  if (with_vel) raw += (size_t)(cap + 1) * 16;
  s.hshift = (float4*)raw;
  raw += HTAB * 16;
  s.hbase = (unsigned*)raw;
  raw += HTAB * 4;
  s.queue = (unsigned short*)raw;
  return s;
}

// coordinate of halo position hx in one dimension: wrapped cell index and the shift s of x_rel = x + s (tile origin
// and periodic image folded into one addend; the addition is exact for own-tile particles)
__device__ __forceinline__ int halo_cell(int c0, int hx, int nc, float L, float o, float& s) {
  int c = c0 + hx - 1;
  if (c < 0) {            // image on the low side: only tiles with c0 == 0, whose origin o is 0
    c += nc;
    s = -L;
  } else if (c >= nc) {   // image on the high side
    c -= nc;
    s = L - o;
  } else {
    s = -o;
  }
  return c;
}

__device__ __forceinline__ float tile_origin(int c0, float edge) { return floorf((float)c0 * edge * 64.0f) * (1.0f / 64.0f); }

// Returns the number of staged particles, or 0xFFFFFFFF if the tile does not fit the shared-memory capacity
// (nothing is staged then).  All threads of the CTA must call it.
template <bool WITH_VEL>
__device__ __forceinline__ unsigned stage_tile(const DevP& p, const TileInfo& T, const float4* __restrict__ pos,
                                               const float4* __restrict__ vel, const TileSmem& sm) {
  const int hxn = T.ex + 2, hyn = T.ey + 2, hzn = T.ez + 2;
  const int nh = hxn * hyn * hzn;
  const float ox = tile_origin(T.c0x, p.edge_x), oy = tile_origin(T.c0y, p.edge_y), oz = tile_origin(T.c0z, p.edge_z);
  for (int h = threadIdx.x; h < nh; h += blockDim.x) {  // one halo cell per thread: where it is, how many, which shift
    const int hx = h % hxn, hy = (h / hxn) % hyn, hz = h / (hxn * hyn);
    float sx, sy, sz;
    const int cx = halo_cell(T.c0x, hx, p.ncx, p.Lx, ox, sx);
    const int cy = halo_cell(T.c0y, hy, p.ncy, p.Ly, oy, sy);
    const int cz = halo_cell(T.c0z, hz, p.ncz, p.Lz, oz, sz);
    const unsigned r = p.cell_rank[((unsigned)cz * p.ncy + cy) * p.ncx + cx];
    const unsigned s = p.cell_start[r];
    sm.hbase[h] = p.cell_start[r + 1] - s;
    sm.hshift[h] = make_float4(sx, sy, sz, u2f(s));
  }
  __syncthreads();
  if (threadIdx.x < 32) {  // exclusive scan of the counts by warp 0
    const int lane = threadIdx.x;
    unsigned run = 0;
    for (int b0 = 0; b0 < nh; b0 += 32) {
      const int h = b0 + lane;
      const unsigned c = h < nh ? sm.hbase[h] : 0u;
      unsigned incl = c;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const unsigned t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
      }
      if (h < nh) sm.hbase[h] = run + incl - c;
      run += __shfl_sync(0xffffffffu, incl, 31);
    }
    if (lane == 0) sm.hbase[nh] = run;
  }
  __syncthreads();
  const unsigned total = sm.hbase[nh];
  if (total > p.tile_cap) return 0xFFFFFFFFu;
  // slot -> halo cell map: one byte per slot, kept in the slot itself until the slot is filled (by the thread that
  // reads the byte); and the slot -> global index offset of every cell
  unsigned char* const cellof = (unsigned char*)sm.spos;
  for (int h = threadIdx.x; h < nh; h += blockDim.x) {
    const unsigned b = sm.hbase[h], e = sm.hbase[h + 1];
    sm.hshift[h].w = u2f(f2u(sm.hshift[h].w) - b);
    for (unsigned k = b; k < e; ++k) cellof[(size_t)k * 16] = (unsigned char)h;
  }
  __syncthreads();
  // one staged slot per thread and iteration (loads of different iterations are independent: several are in flight)
#pragma unroll 4
  for (unsigned sl = threadIdx.x; sl < total; sl += blockDim.x) {
    const float4 sh = sm.hshift[cellof[(size_t)sl * 16]];
    const unsigned g = sl + f2u(sh.w);
    float4 x = pos[g];
    x.x += sh.x;
    x.y += sh.y;
    x.z += sh.z;
    sm.spos[sl] = x;
    if (WITH_VEL) sm.svel[sl] = vel[g];
  }
  if (threadIdx.x == 0) {  // sentinel slot: list padding points here; it is out of range of everything
    sm.spos[p.tile_cap] = make_float4(1e9f, 1e9f, 1e9f, 0.f);
    if (WITH_VEL) sm.svel[p.tile_cap] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  __syncthreads();
  return total;
}

// ----------------------------------------------------------------------------------------------------------------
// Staging recipe.  The per-step passes (density, force) do not rediscover the tile's geometry: at every list build
// k_tile_recipe writes, per tile, a header and one record per RUN of halo cells that is contiguous both in the staged
// image and in the sorted particle arrays (per (y, z) halo row: the cell at x = -1, the tile-aligned cells, the cell
// at x = ex).  Header: x = staged particles (0xFFFFFFFF: tile does not fit), y = runs, z = items | own particles << 16,
// w = first own particle.  Record: x = first global index, y = first staged slot | particles << 16, z = shift code
// cx + 3 cy + 9 cz (per dimension 0 -> -origin, 1 -> -L, 2 -> L - origin), w = index of the run's first item; an ITEM is a
// piece of at most 32 particles of a run: one coalesced load per warp.
// stage_fast: records -> item list in shared memory (one global-memory latency), barrier, every warp copies its
// items in batches of independent loads (one more latency), barrier.  The staged image is bit-identical to stage_tile's.
// ----------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void cp_async16(unsigned dst_smem, const void* src) {  // LDGSTS: no register staging
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst_smem), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

template <bool WITH_VEL>
__device__ __forceinline__ bool stage_fast(const DevP& p, const TileInfo& T, const uint4 hdr, const uint4 R0,
                                           const float4* __restrict__ pos, const float4* __restrict__ vel,
                                           const TileSmem& sm) {
  uint2* const items = (uint2*)sm.hshift;   // [nitems] <= 3 * 36 + tile_cap / 32 <= 2 * HTAB
  float4* const shtab = (float4*)sm.hbase;  // [27] shift of every code
  // R0 = record threadIdx.x, requested by the caller together with the header (whose nruns bounds the records): one
  // latency for both
  const uint4* __restrict__ rec = p.runs + (size_t)blockIdx.x * p.run_stride + 1;
  const unsigned nrec = p.nrun_max;
  const unsigned total = hdr.x, nruns = hdr.y, nitems = hdr.z & 0xFFFFu;
  for (unsigned r = threadIdx.x; r < nrec; r += blockDim.x) {
    const uint4 R = r == threadIdx.x ? R0 : rec[r];
    if (r < nruns && total <= p.tile_cap) {
      const unsigned cnt = R.y >> 16, sb = R.y & 0xFFFFu;
      unsigned io = R.w;
      MDPD_CHECK(p, sb + cnt <= p.tile_cap && R.x + cnt <= p.N && R.z < 27u && R.w + ((cnt + 31u) >> 5) <= 2u * HTAB);
      for (unsigned c = 0; c < cnt; c += 32, ++io)
        items[io] = make_uint2(R.x + c, (sb + c) | ((min(32u, cnt - c) - 1u) << 16) | (R.z << 21));
    }
  }
  if (total > p.tile_cap) return false;  // flagged by k_tile_recipe (block-uniform)
  if (threadIdx.x < 27) {
    const unsigned c = threadIdx.x, cx = c % 3u, cy = (c / 3u) % 3u, cz = c / 9u;
    const float ox = tile_origin(T.c0x, p.edge_x), oy = tile_origin(T.c0y, p.edge_y), oz = tile_origin(T.c0z, p.edge_z);
    shtab[c] = make_float4(cx == 0u ? -ox : (cx == 1u ? -p.Lx : p.Lx - ox), cy == 0u ? -oy : (cy == 1u ? -p.Ly : p.Ly - oy),
                           cz == 0u ? -oz : (cz == 1u ? -p.Lz : p.Lz - oz), 0.f);
  }
  __syncthreads();
  const unsigned warp = threadIdx.x >> 5, lane = threadIdx.x & 31, W = blockDim.x >> 5;
  const unsigned pbase = smem_addr(sm.spos), vbase = smem_addr(sm.svel);
  // asynchronous copies global -> shared of every item of the warp: all in flight at once
  for (unsigned q = warp; q < nitems; q += W) {
    const uint2 it = items[q];
    if (lane <= ((it.y >> 16) & 31u)) {
      const unsigned dst = ((it.y & 0xFFFFu) + lane) << 4;
      cp_async16(pbase + dst, pos + it.x + lane);
      if (WITH_VEL) cp_async16(vbase + dst, vel + it.x + lane);
    }
  }
  cp_async_wait_all();
  __syncwarp();
  // To tile-relative coordinates, in place (a warp touches only what it copied itself).  A tile that does not touch the
  // periodic boundary needs no periodic images: its staged coordinates stay the global ones (differences of nearby
  // fp32 coordinates are as exact as differences of their translates) and the pass over the image is skipped.
  const bool interior = T.c0x > 0 && T.c0x + T.ex < p.ncx && T.c0y > 0 && T.c0y + T.ey < p.ncy && T.c0z > 0 && T.c0z + T.ez < p.ncz;
  for (unsigned q = warp; q < nitems && !interior; q += W) {
    const uint2 it = items[q];
    if (lane <= ((it.y >> 16) & 31u)) {
      const float4 sh = shtab[it.y >> 21];
      float4* const xp = sm.spos + (it.y & 0xFFFFu) + lane;
      float4 x = *xp;
      x.x += sh.x;
      x.y += sh.y;
      x.z += sh.z;
      *xp = x;
    }
  }
  if (threadIdx.x == 0) {  // sentinel slot: list padding points here; it is out of range of everything
    sm.spos[p.tile_cap] = make_float4(1e9f, 1e9f, 1e9f, 0.f);
    if (WITH_VEL) sm.svel[p.tile_cap] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  __syncthreads();
  return true;
}

// stage_bulk: the same staged image by the bulk-copy engine (TMA, 1-D form).  A run of the recipe is contiguous both in
// the sorted arrays and in the staged image, 16-byte aligned on both sides: thread r issues ONE cp.async.bulk
// (global -> shared, completion counted in bytes on an mbarrier) per run and array, thread 0 arms the mbarrier with the
// tile's byte count, everybody waits on its phase.  No per-particle copy instructions, no item list.  The periodic
// shift of a boundary tile is added afterwards, warp per run.  (mdpd_params.flags & MDPD_FLAG_TMA_STAGING; measured
// against stage_fast in profiles/r2_staging.md.)
template <bool WITH_VEL>
__device__ __forceinline__ bool stage_bulk(const DevP& p, const TileInfo& T, const uint4 hdr, const uint4 R0,
                                           const float4* __restrict__ pos, const float4* __restrict__ vel,
                                           const TileSmem& sm) {
  __shared__ __align__(8) unsigned long long mbar;
  uint4* const srec = (uint4*)sm.hshift;    // [nruns] <= 108 <= HTAB
  float4* const shtab = (float4*)sm.hbase;  // [27] shift of every code
  const uint4* __restrict__ rec = p.runs + (size_t)blockIdx.x * p.run_stride + 1;
  const unsigned total = hdr.x, nruns = hdr.y;
  if (total > p.tile_cap) return false;  // flagged by k_tile_recipe (block-uniform)
  const unsigned mb = smem_addr(&mbar);
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mb) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  if (threadIdx.x < 27) {
    const unsigned c = threadIdx.x, cx = c % 3u, cy = (c / 3u) % 3u, cz = c / 9u;
    const float ox = tile_origin(T.c0x, p.edge_x), oy = tile_origin(T.c0y, p.edge_y), oz = tile_origin(T.c0z, p.edge_z);
    shtab[c] = make_float4(cx == 0u ? -ox : (cx == 1u ? -p.Lx : p.Lx - ox), cy == 0u ? -oy : (cy == 1u ? -p.Ly : p.Ly - oy),
                           cz == 0u ? -oz : (cz == 1u ? -p.Lz : p.Lz - oz), 0.f);
  }
  __syncthreads();
  const unsigned pbase = smem_addr(sm.spos), vbase = smem_addr(sm.svel);
  for (unsigned r = threadIdx.x; r < nruns; r += blockDim.x) {
    const uint4 R = r == threadIdx.x ? R0 : rec[r];  // R0: requested by the caller together with the header
    srec[r] = R;
    const unsigned cnt = R.y >> 16, sb = R.y & 0xFFFFu;
    MDPD_CHECK(p, sb + cnt <= p.tile_cap && R.x + cnt <= p.N && R.z < 27u && r < (unsigned)HTAB);
    if (cnt) {
      asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(pbase + (sb << 4)),
                   "l"(pos + R.x), "r"(cnt << 4), "r"(mb)
                   : "memory");
      if (WITH_VEL)
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(vbase + (sb << 4)),
                     "l"(vel + R.x), "r"(cnt << 4), "r"(mb)
                     : "memory");
    }
  }
  if (threadIdx.x == 0)
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mb), "r"((total << 4) * (WITH_VEL ? 2u : 1u)) : "memory");
  {
    unsigned done = 0;
    while (!done)
      asm volatile(
          "{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0; selp.u32 %0, 1, 0, p; }" : "=r"(done) : "r"(mb) : "memory");
  }
  const bool interior = T.c0x > 0 && T.c0x + T.ex < p.ncx && T.c0y > 0 && T.c0y + T.ey < p.ncy && T.c0z > 0 && T.c0z + T.ez < p.ncz;
  if (!interior) {  // to tile-relative coordinates, in place, warp per run
    __syncthreads();  // the run records
    const unsigned warp = threadIdx.x >> 5, lane = threadIdx.x & 31, W = blockDim.x >> 5;
    for (unsigned r = warp; r < nruns; r += W) {
      const uint4 R = srec[r];
      const unsigned cnt = R.y >> 16, sb = R.y & 0xFFFFu;
      const float4 sh = shtab[R.z];
      for (unsigned c = lane; c < cnt; c += 32) {
        float4* const xp = sm.spos + sb + c;
        float4 x = *xp;
        x.x += sh.x;
        x.y += sh.y;
        x.z += sh.z;
        *xp = x;
      }
    }
  }
  if (threadIdx.x == 0) {  // sentinel slot: list padding points here; it is out of range of everything
    sm.spos[p.tile_cap] = make_float4(1e9f, 1e9f, 1e9f, 0.f);
    if (WITH_VEL) sm.svel[p.tile_cap] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  __syncthreads();
  return true;
}

// ----------------------------------------------------------------------------------------------------------------
// Tile recipe.  After every sort k_tile_recipe (one CTA per tile) writes what the tile passes need to stage the tile
// without rediscovering its geometry: the header and run records described above, and the table of the first
// staged slot of every halo cell (16-bit, nh + 1 entries, at uint4 offset hb_off of the tile's record).  It also
// keeps the two occupancy maxima (tile + halo: shared-memory capacity; tile alone: CTA size).
// ----------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_tile_recipe(const DevP p, int latch_faults) {
  if (!p.ctl->rebuild) return;
  __shared__ unsigned s_hb[HTAB];  // particles of every halo cell, then their exclusive scan (first staged slot)
  __shared__ unsigned s_g[HTAB];   // first sorted (global) index of every halo cell
  const TileInfo T = p.tiles[blockIdx.x];
  const int hxn = T.ex + 2, hyn = T.ey + 2, hzn = T.ez + 2;
  const int nh = hxn * hyn * hzn;
  for (int h = threadIdx.x; h < nh; h += blockDim.x) {
    const int hx = h % hxn, hy = (h / hxn) % hyn, hz = h / (hxn * hyn);
    float a;
    const int cx = halo_cell(T.c0x, hx, p.ncx, 0.f, 0.f, a), cy = halo_cell(T.c0y, hy, p.ncy, 0.f, 0.f, a),
              cz = halo_cell(T.c0z, hz, p.ncz, 0.f, 0.f, a);
    const unsigned r = p.cell_rank[((unsigned)cz * p.ncy + cy) * p.ncx + cx];
    const unsigned s = p.cell_start[r];
    s_hb[h] = p.cell_start[r + 1] - s;
    s_g[h] = s;
  }
  __syncthreads();
  const int lane = threadIdx.x & 31;
  if (threadIdx.x < 32) {  // exclusive scan of the counts by warp 0
    unsigned run = 0;
    for (int b0 = 0; b0 < nh; b0 += 32) {
      const int h = b0 + lane;
      const unsigned c = h < nh ? s_hb[h] : 0u;
      unsigned incl = c;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const unsigned t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
      }
      if (h < nh) s_hb[h] = run + incl - c;
      run += __shfl_sync(0xffffffffu, incl, 31);
    }
    if (lane == 0) s_hb[nh] = run;
  }
  __syncthreads();
  const unsigned total = s_hb[nh];
  const bool fits = total <= p.tile_cap;
  const unsigned own_s = p.cell_start[T.rank0], own_n = p.cell_start[T.rank0 + T.ncell_own] - own_s;
  uint4* const out = p.runs + (size_t)blockIdx.x * p.run_stride;
  unsigned short* const hb16 = (unsigned short*)(out + p.hb_off);
  for (int h = threadIdx.x; h <= nh; h += blockDim.x) hb16[h] = (unsigned short)min(s_hb[h], 0xFFFFu);
  if (threadIdx.x < 32) {  // run records: per (y, z) halo row the cell at x = -1, the tile-aligned cells, the cell at x = ex
    const unsigned nruns = 3u * hyn * hzn;
    unsigned run_items = 0;
    for (unsigned r0 = 0; r0 < nruns; r0 += 32) {
      const unsigned r = r0 + lane;
      unsigned cnt = 0, sb = 0, g = 0, code = 0;
      if (r < nruns) {
        const int seg = r % 3, hy = (r / 3) % hyn, hz = r / (3 * hyn);
        const int hx = seg == 0 ? 0 : (seg == 1 ? 1 : hxn - 1), len = seg == 1 ? T.ex : 1;
        const int h0 = (hz * hyn + hy) * hxn + hx;
        sb = s_hb[h0];
        cnt = s_hb[h0 + len] - sb;
        g = s_g[h0];
        const int cx = T.c0x + hx - 1, cy = T.c0y + hy - 1, cz = T.c0z + hz - 1;
        code = (cx < 0 ? 1u : (cx >= p.ncx ? 2u : 0u)) + 3u * (cy < 0 ? 1u : (cy >= p.ncy ? 2u : 0u)) +
               9u * (cz < 0 ? 1u : (cz >= p.ncz ? 2u : 0u));
      }
      const unsigned nit = (cnt + 31u) >> 5;
      unsigned incl = nit;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const unsigned t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
      }
      if (r < nruns) out[1 + r] = make_uint4(g, sb | (cnt << 16), code, run_items + incl - nit);
      run_items += __shfl_sync(0xffffffffu, incl, 31);
    }
    if (lane == 0) {
      out[0] = fits ? make_uint4(total, nruns, run_items | (own_n << 16), own_s) : make_uint4(0xFFFFFFFFu, 0u, own_n << 16, own_s);
      atomicMax(&p.ctl->max_halo, total);
      atomicMax(&p.ctl->max_own, own_n);
      if (!fits && latch_faults) {  // reported as MDPD_EOVERFLOW; the tile passes skip this tile
        atomicOr(&p.ctl->err, ERR_TILE);
        atomicAdd(&p.ctl->overflow, 1ull);
      }
    }
  }
}

// Record threadIdx.x of this tile's staging recipe (requested together with the header), and L2 prefetches of the recipe
// of the tile that starts one CTA lifetime later (CTAs start in blockIdx order; `ahead` = resident CTAs of the grid).
__device__ __forceinline__ uint4 first_record(const DevP& p, const unsigned ahead) {
  const uint4* __restrict__ rec = p.runs + (size_t)blockIdx.x * p.run_stride + 1;
  const uint4 R0 = threadIdx.x < p.nrun_max ? rec[threadIdx.x] : make_uint4(0u, 0u, 0u, 0u);
  const unsigned nb = blockIdx.x + ahead;
  if (nb < gridDim.x && threadIdx.x * 8u < p.run_stride) prefetch_l2(p.runs + (size_t)nb * p.run_stride + threadIdx.x * 8u);
  return R0;
}
// ... and of its hand-out records and first list chunks (`hdrn` = that tile's header, requested at the start of the CTA,
// used when the own tile has been staged: nobody waits for it)
__device__ __forceinline__ void prefetch_handout(const DevP& p, const unsigned ahead, const uint4 hdrn, const uint2* __restrict__ info,
                                                 const uint4* __restrict__ lst) {
  if (blockIdx.x + ahead >= gridDim.x) return;
  const unsigned osn = hdrn.w, nownn = hdrn.z >> 16;
  if (threadIdx.x * 16u < nownn) prefetch_l2(info + osn + threadIdx.x * 16u);  // 128-byte lines: 16 records, 8 chunks
  for (unsigned t = threadIdx.x * 8u; t < nownn; t += blockDim.x * 8u) prefetch_l2(lst + osn + t);
}

// group of 32 sorted own particles that warp `warp` of W takes in its round r (see the hand-out below)
__device__ __forceinline__ unsigned group_of_round(unsigned r, unsigned warp, unsigned W) {
  return (r & 1u) ? (r + 1u) * W - 1u - warp : r * W + warp;
}

// ----------------------------------------------------------------------------------------------------------------
// a3 (and S8f f1): k_cells -- neighbours straight from the cells.  One kernel, two uses:
//   MODE 0  Verlet list build (full list: every j != i with r < rc + skin at build time), in the rebuild chain;
//   MODE 1  the list-free path (mdpd_params.flags & MDPD_FLAG_DIRECT): every step, the in-range (r < rc) lists of
//           the step straight from the 27-cell stencil, the density pass over them, and the hand-out of the force pass.
//
// Orientation: LANE = CANDIDATE, the own particle is broadcast.  A warp takes a pair of x-adjacent own cells, one cell
// at a time.  The candidates of a cell (the particles of its 27-cell stencil: nine contiguous runs of the staged image,
// one per (y, z) row of halo cells) are flattened and held IN REGISTERS, 32 per chunk, up to CHMAX chunks at a time:
// per candidate (x, y, z, |x|^2) in tile-CENTRED coordinates and its staged slot.  The warp then loops over the cell's
// own particles: one uniform 16-byte shared-memory load of x_i (amortised over all chunks), and per chunk the range test
// in dot-product form
//     |xc|^2 - 2 xi . xc  <  cut^2 - |xi|^2          (3 FFMA + 1 compare per 32 candidates),
// evaluated with a slack `dot_margin` on cut^2 that covers its rounding error (|x| <= ~4 in centred coordinates): the
// hits are a SUPERSET of the exact r^2 < cut^2 set.  The hits of a chunk go straight into the particle's row of a
// per-warp row buffer in shared memory: ballot, rank of the lane among the hits (popc of the ballot below the lane),
// one predicated 16-bit store of the candidate's slot.  No hit masks, no decoding pass; entries come out in increasing
// candidate (= staged-slot) order: deterministic.  (A first version with LANE = own particle and the candidate
// broadcast had an even simpler loop but is bound by the 512 bytes every warp-wide 16-byte load returns to the
// registers: 13.1 ms against 11.4 ms of round 1's kernel on config 4a; profiles/r2_cells.md.)
// When the rows of the pair are complete, lane = row:
// MODE 0 copies the rows to the list (16-byte chunks, layout [chunk][particle]: consecutive lanes write consecutive
// particles).  MODE 1 walks its row with the EXACT fp32 distance (same arithmetic as k_density): density sum over
// r < rd; entries that fail 1e-12 < r^2 < rc^2 exactly (slack hits, coincident particles R10, frozen-frozen pairs R8)
// are replaced by the far-away sentinel slot, and the row becomes the step's compact list.
// ----------------------------------------------------------------------------------------------------------------
#ifndef CELLS_W0
#define CELLS_W0 8
#endif
constexpr int CELLS_MAXW0 = CELLS_W0;  // most warps per CTA of the list build (two resident CTAs: 65536 / (64 W) registers per thread)
constexpr int CELLS_MAXW = 8;          // ... of the list-free pass
constexpr int CHMAX = 12;             // candidate chunks (of 32) held in registers at a time: one window
constexpr unsigned ROW_SLACK = 40;    // row capacity beyond the list capacity: the saturated count (cap + 1) plus one chunk's worth of hits

__host__ __device__ inline unsigned cells_row_bytes(unsigned rowcap) {
  unsigned b = 2u * (rowcap + ROW_SLACK) + 16u;  // + one chunk of sentinel padding
  if (((b >> 4) & 1u) == 0u) b += 16u;           // odd number of 16-byte groups: 16-byte row reads of consecutive lanes do not collide
  return b;
}
constexpr unsigned CELLS_ROW0_BYTES = 32 * CHMAX * 2 + 16;  // list build: one row per warp, a whole window of hits
// per_warp: bytes of row buffer per warp (list build: CELLS_ROW0_BYTES; list-free pass: 32 rows + their entry counts)
__host__ __device__ inline size_t cells_smem_bytes(unsigned tile_cap, size_t per_warp, unsigned nwarps) {
  return (size_t)(tile_cap + 1) * 16 + HTAB * 16 + HTAB * 4 + HTAB * 2 + (size_t)nwarps * per_warp;
}

__device__ __forceinline__ void sts_u16(unsigned addr, unsigned v) {
  asm volatile("st.shared.u16 [%0], %1;" ::"r"(addr), "h"((unsigned short)v) : "memory");
}
__device__ __forceinline__ uint4 lds4u(unsigned addr) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
  return v;
}

// stage_fast's copy (recipe -> items -> cp.async), then one pass in place to centred coordinates and |x|^2 (bit 0 of
// which carries the frozen flag when HAS_WALL); also fetches the tile's table of first staged slots.
template <bool HAS_WALL>
__device__ __forceinline__ bool stage_cells(const DevP& p, const TileInfo& T, const uint4 hdr, const float4* __restrict__ pos,
                                            float4* img, uint2* items, float4* shtab, unsigned short* hb) {
  const uint4* __restrict__ rcp = p.runs + (size_t)blockIdx.x * p.run_stride;
  const uint4* __restrict__ rec = rcp + 1;
  const unsigned nrec = p.nrun_max;
  const unsigned total = hdr.x, nruns = hdr.y, nitems = hdr.z & 0xFFFFu;
  if (total > p.tile_cap) return false;  // flagged by k_tile_recipe (block-uniform)
  for (unsigned r = threadIdx.x; r < nrec; r += blockDim.x) {
    const uint4 R = rec[r];
    if (r < nruns) {
      const unsigned cnt = R.y >> 16, sb = R.y & 0xFFFFu;
      unsigned io = R.w;
      MDPD_CHECK(p, sb + cnt <= p.tile_cap && R.x + cnt <= p.N && R.z < 27u && R.w + ((cnt + 31u) >> 5) <= 2u * HTAB);
      for (unsigned c = 0; c < cnt; c += 32, ++io)
        items[io] = make_uint2(R.x + c, (sb + c) | ((min(32u, cnt - c) - 1u) << 16) | (R.z << 21));
    }
  }
  {
    const unsigned nh1 = (unsigned)((T.ex + 2) * (T.ey + 2) * (T.ez + 2)) + 1u;
    const uint4* __restrict__ src = rcp + p.hb_off;
    uint4* const dst = (uint4*)hb;
    for (unsigned q = threadIdx.x; q < (nh1 + 7u) / 8u; q += blockDim.x) dst[q] = src[q];
  }
  if (threadIdx.x < 27) {  // shift of every periodic-image code, minus the tile centre (both on the 2^-6 grid)
    const unsigned c = threadIdx.x, cx = c % 3u, cy = (c / 3u) % 3u, cz = c / 9u;
    const float ox = tile_origin(T.c0x, p.edge_x), oy = tile_origin(T.c0y, p.edge_y), oz = tile_origin(T.c0z, p.edge_z);
    const float hx = floorf(0.5f * (float)T.ex * p.edge_x * 64.0f) * (1.0f / 64.0f),
                hy = floorf(0.5f * (float)T.ey * p.edge_y * 64.0f) * (1.0f / 64.0f),
                hz = floorf(0.5f * (float)T.ez * p.edge_z * 64.0f) * (1.0f / 64.0f);
    shtab[c] = make_float4((cx == 0u ? -ox : (cx == 1u ? -p.Lx : p.Lx - ox)) - hx, (cy == 0u ? -oy : (cy == 1u ? -p.Ly : p.Ly - oy)) - hy,
                           (cz == 0u ? -oz : (cz == 1u ? -p.Lz : p.Lz - oz)) - hz, 0.f);
  }
  __syncthreads();
  const unsigned warp = threadIdx.x >> 5, lane = threadIdx.x & 31, W = blockDim.x >> 5;
  const unsigned ibase = smem_addr(img);
  for (unsigned q = warp; q < nitems; q += W) {
    const uint2 it = items[q];
    if (lane <= ((it.y >> 16) & 31u)) cp_async16(ibase + (((it.y & 0xFFFFu) + lane) << 4), pos + it.x + lane);
  }
  cp_async_wait_all();
  __syncwarp();
  for (unsigned q = warp; q < nitems; q += W) {  // a warp touches only what it copied itself
    const uint2 it = items[q];
    if (lane <= ((it.y >> 16) & 31u)) {
      const float4 sh = shtab[it.y >> 21];
      float4* const xp = img + (it.y & 0xFFFFu) + lane;
      float4 x = *xp;
      x.x += sh.x;
      x.y += sh.y;
      x.z += sh.z;
      float q2 = fmaf(x.z, x.z, fmaf(x.y, x.y, x.x * x.x));
      if (HAS_WALL) q2 = u2f((f2u(q2) & ~1u) | (f2u(x.w) >> 31));
      x.w = q2;
      *xp = x;
    }
  }
  if (threadIdx.x == 0) img[p.tile_cap] = make_float4(1e9f, 1e9f, 1e9f, 3e18f);  // sentinel slot: out of range of everything
  __syncthreads();
  return true;
}

struct CandRegs {  // one window of candidates: chunk t, this lane
  float x[CHMAX], y[CHMAX], z[CHMAX], q[CHMAX];
  unsigned s[CHMAX];  // staged slot (the sentinel past the end)
};

// own particles [il0, il1) of the cell whose first staged slot is S_cell, against the NCH chunks of the window; particle
// il appends its hits to row row0 + (il - il0) of the warp's row buffer.  All lanes must call it.  (List-free pass.)
template <int NCH>
__device__ __forceinline__ void cell_tests(const DevP& p, const CandRegs& C, const float4* img, const unsigned S_cell, const unsigned il0,
                                           const unsigned il1, const unsigned row0, const unsigned rbase_w,
                                           const unsigned row_bytes, unsigned short* rowcnt, const float cut2,
                                           const unsigned rowcap, const unsigned ltmask, const unsigned lane) {
  float4 xi = img[S_cell + il0];
  for (unsigned il = il0; il < il1; ++il) {
    const float ax = -2.0f * xi.x, ay = -2.0f * xi.y, az = -2.0f * xi.z;
    const float thr = cut2 - fmaf(xi.z, xi.z, fmaf(xi.y, xi.y, xi.x * xi.x));
    const unsigned self = S_cell + il;
    const unsigned row = row0 + (il - il0);
    const unsigned ra = rbase_w + row * row_bytes;
    // running write address of the row; it saturates at rowcap + 1 entries: a list that stays within rowcap is never
    // clamped, a longer one reads back as rowcap + 1 (an overflow), and no store leaves the row (rowcap + 40 entries)
    const unsigned lim = ra + 2u * rowcap + 2u;
    unsigned na = ra + 2u * rowcnt[row];
    xi = img[S_cell + min(il + 1u, il1 - 1u)];  // next particle's position in flight
#pragma unroll
    for (int t = 0; t < NCH; ++t) {
      const float v = fmaf(C.x[t], ax, fmaf(C.y[t], ay, fmaf(C.z[t], az, C.q[t])));
      const bool hit = v < thr && C.s[t] != self;
      const unsigned b = __ballot_sync(0xffffffffu, hit);
      MDPD_CHECK(p, na + 2u * __popc(b) <= ra + row_bytes - 16u && row < 32u);
      if (hit) sts_u16(na + 2u * __popc(b & ltmask), C.s[t]);
      na = min(na + 2u * __popc(b), lim);
    }
    if (lane == 0) rowcnt[row] = (unsigned short)((na - ra) >> 1);
    __syncwarp();  // orders this store before the re-read of rowcnt[row] by all lanes in the next window's call
  }
}

// List build: the same tests, but a particle's row is complete when its chunk loop ends, so it is copied to the list
// right away (lane c copies the 16-byte chunk c) and the warp needs ONE row, sized for a whole window of hits: no
// clamping, and the shared memory it frees buys resident warps.  `ra` = shared address of the warp's row (16-byte
// aligned), gi0 = sorted index of particle il0.  FIRST / LAST: this window is the first / last of the cell's stencil
// (both true unless the stencil holds more than 32 CHMAX particles; then the caller loops particle by particle over
// the windows and `n0` carries the row's fill from window to window).  Statistics are kept by lane 0.
// SELF0: the cell's own particles are the first candidates of the window (flat index = index in the cell) and the
// cell holds at most 32: the particle itself is lane il of chunk 0, nowhere else.
template <int NCH, bool FIRST, bool LAST, bool SELF0>
__device__ __forceinline__ void cell_tests_flush(const DevP& p, const CandRegs& C, const float4* img, const unsigned S_cell,
                                                 const unsigned il0, const unsigned il1, const unsigned gi0, const unsigned ra,
                                                 const float cut2, const unsigned ltmask, const unsigned lane,
                                                 unsigned* lhist, unsigned& smax, unsigned& ssum, bool& sover, unsigned& n0) {
  const unsigned sent2 = p.tile_cap | (p.tile_cap << 16);
  const unsigned fill = (p.cap + 8u + 7u) >> 3;  // chunks that can reach the list, plus one of padding
  float4 xi = img[S_cell + il0];
  unsigned myn = 0;  // lane k: list length of particle il0 + k (il1 - il0 <= 32)
  for (unsigned il = il0; il < il1; ++il) {
    const float ax = -2.0f * xi.x, ay = -2.0f * xi.y, az = -2.0f * xi.z;
    const float thr = cut2 - fmaf(xi.z, xi.z, fmaf(xi.y, xi.y, xi.x * xi.x));
    const unsigned self = S_cell + il;
    xi = img[S_cell + min(il + 1u, il1 - 1u)];  // next particle's position in flight
    if (FIRST) {  // fresh row: sentinel everywhere a flushed chunk can look (the hits overwrite it)
      if (lane < fill) asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(ra + 16u * lane), "r"(sent2) : "memory");
      __syncwarp();
    }
    unsigned na = ra + 2u * (FIRST ? 0u : n0);
#pragma unroll
    for (int t = 0; t < NCH; ++t) {
      const float v = fmaf(C.x[t], ax, fmaf(C.y[t], ay, fmaf(C.z[t], az, C.q[t])));
      bool hit = v < thr;
      if (SELF0) {
        if (t == 0) hit = hit && lane != il;
      } else {
        hit = hit && C.s[t] != self;
      }
      const unsigned b = __ballot_sync(0xffffffffu, hit);
      MDPD_CHECK(p, na + 2u * __popc(b) <= ra + CELLS_ROW0_BYTES);
      if (hit) sts_u16(na + 2u * __popc(b & ltmask), C.s[t]);
      na += 2u * __popc(b);
      // A single window (FIRST && LAST) cannot outgrow the row: 32 NCH - 1 hits at most.  When the fill is carried
      // from window to window it can (a collapsed cluster, many coincident particles: R10 allows them), so there the
      // write address saturates one chunk short of the row's end: 360 entries, far above any capacity (<= 128), so a
      // saturated row still reads as an overflow below, and no store leaves the row.
      if (!(FIRST && LAST)) na = min(na, ra + CELLS_ROW0_BYTES - 64u);
    }
    __syncwarp();
    unsigned n = (na - ra) >> 1;
    n0 = n;
    MDPD_CHECK(p, gi0 + (il - il0) < p.N && S_cell + il < p.tile_cap);
    if (LAST) {
      if (n > p.cap) n = 0xFFFFu;  // overflow marker
      if (lane < (((n > p.cap ? 0u : n) + 7u) >> 3)) p.nbr[(size_t)lane * p.N + gi0 + (il - il0)] = lds4u(ra + 16u * lane);
      if (lane == il - il0) myn = n;
      __syncwarp();
    }
  }
  if (LAST && lane < il1 - il0) {  // lane = particle: lengths, own slots, histogram of the hand-out sort, statistics
    const bool over = myn > p.cap;
    if (over) myn = 0;  // reported as MDPD_EOVERFLOW; this particle's list is emptied
    p.nnbr[gi0 + lane] = myn;
    p.self_loc[gi0 + lane] = (unsigned short)(S_cell + il0 + lane);
    atomicAdd(&lhist[LCAP - min(myn, LCAP)], 1u);
    smax = max(smax, myn);
    ssum += myn;
    sover = sover || over;
  }
}

template <bool HAS_WALL, bool ALL>
__device__ __forceinline__ void direct_entry(const DevP& p, const unsigned ibase, const float4 xi, const unsigned walli,
                                             const unsigned j, const unsigned kaddr, const unsigned sent, float& rho,
                                             unsigned& nin) {
  MDPD_CHECK(p, j <= p.tile_cap);
  const float4 xj = lds4(ibase + (j << 4));  // padding entries hit the far-away sentinel
  const float dx = xi.x - xj.x, dy = xi.y - xj.y, dz = xi.z - xj.z;
  const float r2 = dx * dx + dy * dy + dz * dz;
  const float w = __saturatef(fmaf(-sqrt_fast(r2), p.inv_rd, 1.0f));  // 1 at r = 0 (coincident particles, R10)
  rho = fmaf(w, w, rho);
  bool in = f2u(r2 - 1e-12f) < f2u(p.rc2 - 1e-12f);  // 1e-12 < r2 < rc2, exact (see density_entry)
  if (HAS_WALL && ALL) in = in && !(walli & f2u(xj.w) & 1u);  // frozen-frozen pairs do not interact (R8)
  if (!in) sts_u16(kaddr, sent);
  nin += in ? 1u : 0u;
}

template <int MODE, bool HAS_WALL, bool ALL>
__global__ void __launch_bounds__((MODE ? CELLS_MAXW : CELLS_MAXW0) * 32, 2) k_cells(const DevP p, int always) {
  if (!always && !p.ctl->rebuild) return;
  extern __shared__ __align__(16) unsigned char smraw[];
  float4* const img = (float4*)smraw;
  unsigned char* q = smraw + (size_t)(p.tile_cap + 1) * 16;
  uint2* const sitems = (uint2*)q;                    // staging items; afterwards the histogram
  unsigned* const lhist = (unsigned*)q;               // [LCAP + 1] bins (bin 0 = longest), then: max, sum, faults, next item
  q += HTAB * 16;
  float4* const shtab = (float4*)q;
  q += HTAB * 4;
  unsigned short* const hb = (unsigned short*)q;
  q += HTAB * 2;
  const unsigned cur = p.ctl->cur;
  const TileInfo T = p.tiles[blockIdx.x];
  const uint4 hdr = p.runs[(size_t)blockIdx.x * p.run_stride];
  const unsigned os = hdr.w, nown = hdr.z >> 16;
  const unsigned warp = threadIdx.x >> 5, lane = threadIdx.x & 31, W = blockDim.x >> 5;
  if (!stage_cells<HAS_WALL>(p, T, hdr, p.pos[cur], img, sitems, shtab, hb)) {  // does not fit: empty lists, the passes skip the tile
    for (unsigned t = threadIdx.x; t < nown; t += blockDim.x) {
      if (MODE == 0) {
        p.nnbr[os + t] = 0u;
        p.self_loc[os + t] = 0;
      } else {
        p.nact[os + t] = 0;
      }
    }
    return;
  }
  for (unsigned k = threadIdx.x; k < LCAP + 8u; k += blockDim.x) lhist[k] = 0u;
  __syncthreads();
  const int hxn = T.ex + 2, hyn = T.ey + 2;
  const unsigned rowcap = p.cap_act, row_bytes = p.rows_direct;  // MODE 1: 32 rows per warp
  const float cut2 = (MODE ? p.rc2 : p.rlist2) + p.dot_margin;
  const unsigned sent = p.tile_cap;
  const unsigned ibase = smem_addr(img);
  // MODE 0: one row per warp (a window's worth of hits); MODE 1: 32 rows per warp and their entry counts
  unsigned short* const rowcnt = (unsigned short*)(q + (size_t)W * 32 * row_bytes) + warp * 32;
  const unsigned rbase_w = smem_addr(q) + warp * (MODE ? 32u * row_bytes : CELLS_ROW0_BYTES);
  const unsigned rbase = rbase_w + lane * row_bytes;  // MODE 1: the row this lane flushes
  const unsigned ltmask = (1u << lane) - 1u;
  const uint4* __restrict__ rec = p.runs + (size_t)blockIdx.x * p.run_stride + 1;
  unsigned smax = 0, ssum = 0;
  bool sover = false;
  float4* __restrict__ vel = p.vel[cur];
  // MODE 1, rows in use: lane = row; which particle the row belongs to
  unsigned rows_used = 0, my_gi = 0, my_self = 0;

  auto flush = [&]() {
    __syncwarp();
    const bool active = lane < rows_used;
    unsigned cnt = active ? rowcnt[lane] : 0u;
    const bool over = cnt > rowcap;
    if (over) cnt = 0;  // reported as MDPD_EOVERFLOW; this particle's list is emptied
    if (active)
      for (unsigned k = cnt; k & 7u; ++k) sts_u16(rbase + 2u * k, sent);  // pad the last chunk with the sentinel
    __syncwarp();
    const unsigned nch = (cnt + 7u) >> 3;
    const unsigned wch = __reduce_max_sync(0xffffffffu, nch);
    const float4 xi = img[active ? my_self : sent];
    const unsigned walli = HAS_WALL ? (f2u(xi.w) & 1u) : 0u;
    float rho = 0.0f;
    unsigned nin = 0;
    for (unsigned c = 0; c < nch; ++c) {
      const unsigned ka = rbase + 16u * c;
      const uint4 e = lds4u(ka);
      direct_entry<HAS_WALL, ALL>(p, ibase, xi, walli, e.x & 0xFFFFu, ka, sent, rho, nin);
      direct_entry<HAS_WALL, ALL>(p, ibase, xi, walli, e.x >> 16, ka + 2u, sent, rho, nin);
      direct_entry<HAS_WALL, ALL>(p, ibase, xi, walli, e.y & 0xFFFFu, ka + 4u, sent, rho, nin);
      direct_entry<HAS_WALL, ALL>(p, ibase, xi, walli, e.y >> 16, ka + 6u, sent, rho, nin);
      direct_entry<HAS_WALL, ALL>(p, ibase, xi, walli, e.z & 0xFFFFu, ka + 8u, sent, rho, nin);
      direct_entry<HAS_WALL, ALL>(p, ibase, xi, walli, e.z >> 16, ka + 10u, sent, rho, nin);
      direct_entry<HAS_WALL, ALL>(p, ibase, xi, walli, e.w & 0xFFFFu, ka + 12u, sent, rho, nin);
      direct_entry<HAS_WALL, ALL>(p, ibase, xi, walli, e.w >> 16, ka + 14u, sent, rho, nin);
    }
    __syncwarp();
    for (unsigned c = 0; c < wch; ++c)
      if (c < nch) p.act[(size_t)c * p.N + my_gi] = lds4u(rbase + 16u * c);
    if (active) {
      p.nact[my_gi] = (unsigned short)cnt;
      vel[my_gi].w = rho * p.Krho;
      const unsigned fy = (HAS_WALL && !ALL && walli) ? 0x80000000u : cnt;  // frozen: force not needed (R8)
      p.dinfo[my_gi] = make_uint2((my_gi - os) | (my_self << 16), fy);     // unsorted; the tail below orders them
      atomicAdd(&lhist[LCAP - min(fy & 0x7FFFFFFFu, LCAP)], 1u);
      ssum += nin;
      sover = sover || over;
    }
    __syncwarp();
    rows_used = 0;
  };

  // work items: pairs of x-adjacent own cells, handed out through a counter in shared memory
  const unsigned xpairs = ((unsigned)T.ex + 1u) >> 1, nitems = xpairs * (unsigned)(T.ey * T.ez);
  for (;;) {
    unsigned it = 0;
    if (lane == 0) it = atomicAdd(&lhist[LCAP + 4], 1u);
    it = __shfl_sync(0xffffffffu, it, 0);
    if (it >= nitems) break;
    const int xp = (int)(it % xpairs), rowi = (int)(it / xpairs);
    const int hy = 1 + rowi % T.ey, hz = 1 + rowi / T.ey;
    const int h0 = (hz * hyn + hy) * hxn + 1;  // halo index of the row's first own cell
    const unsigned g_row = rec[(unsigned)(hz * hyn + hy) * 3u + 1u].x, sb_row = hb[h0];
    for (int cx = 2 * xp; cx < min(2 * xp + 2, T.ex); ++cx) {
      const unsigned S_cell = hb[h0 + cx], n = (unsigned)hb[h0 + cx + 1] - S_cell, G_cell = g_row + (S_cell - sb_row);
      if (n == 0) continue;
      // the candidate runs, lane r < 11 holds run r: the cell itself first (so that a particle finds itself at lane il of
      // chunk 0), then the (dz, dy) rows of the stencil, three cells each, the centre row as its left and right cell;
      // inclusive scan of the run lengths
      unsigned run_b = 0, run_n = 0;
      if (lane < 11) {
        const int q9 = lane == 0 ? 4 : (lane <= 4 ? (int)lane - 1 : (lane <= 6 ? 4 : (int)lane - 2));  // the row of run `lane`
        const int hrow = ((hz - 1 + q9 / 3) * hyn + (hy - 1 + q9 % 3)) * hxn + cx;  // halo x of cell cx - 1
        run_b = hb[hrow];
        run_n = (unsigned)hb[hrow + 3] - run_b;
        if (lane == 0) { run_b = S_cell; run_n = n; }
        if (lane == 5) run_n = S_cell - run_b;
        if (lane == 6) { run_n = run_b + run_n - (S_cell + n); run_b = S_cell + n; }
      }
      unsigned incl = run_n;
#pragma unroll
      for (int o = 1; o < 16; o <<= 1) {
        const unsigned t = __shfl_up_sync(0xffffffffu, incl, o);
        if ((int)lane >= o) incl += t;
      }
      const unsigned ncand = __shfl_sync(0xffffffffu, incl, 10);
      const unsigned run_o = incl - run_n;  // exclusive offset of the lane's run
      unsigned rend[10];
#pragma unroll
      for (int r = 0; r < 10; ++r) rend[r] = __shfl_sync(0xffffffffu, incl, r);
      CandRegs C;
      // one window of candidates into registers: flat candidate index -> staged slot (past the end: the sentinel, never hit)
      auto load_window = [&](const unsigned win, const unsigned nch) {
#pragma unroll
        for (int t = 0; t < CHMAX; ++t) {
          if ((unsigned)t < nch) {  // warp-uniform
            const unsigned f = win + 32u * t + lane;
            unsigned r = 0;
#pragma unroll
            for (int qq = 0; qq < 10; ++qq) r += (f >= rend[qq]) ? 1u : 0u;
            const unsigned rb = __shfl_sync(0xffffffffu, run_b, r), ro = __shfl_sync(0xffffffffu, run_o, r);
            const unsigned cs = f < ncand ? rb + (f - ro) : sent;
            MDPD_CHECK(p, cs <= p.tile_cap && r <= 10u);
            const float4 xc = img[cs];
            C.x[t] = xc.x;
            C.y[t] = xc.y;
            C.z[t] = xc.z;
            C.q[t] = xc.w;
            C.s[t] = cs;
          }
        }
      };
      if (MODE == 0) {
        unsigned n0 = 0;
        if (ncand <= 32u * CHMAX) {  // the whole stencil fits one window: particle after particle, each flushed at once
          const unsigned nch = (ncand + 31u) >> 5;
          load_window(0u, nch);
          for (unsigned r0 = 0; r0 < n; r0 += 32u) {
            const unsigned r1 = min(n, r0 + 32u);
#define CELLS_CASE(K)                                                                                                              \
  case K:                                                                                                                            \
    if (n <= 32u)                                                                                                                    \
      cell_tests_flush<K, true, true, true>(p, C, img, S_cell, r0, r1, G_cell + r0, rbase_w, cut2, ltmask, lane, lhist, smax, ssum,  \
                                            sover, n0);                                                                              \
    else                                                                                                                             \
      cell_tests_flush<K, true, true, false>(p, C, img, S_cell, r0, r1, G_cell + r0, rbase_w, cut2, ltmask, lane, lhist, smax, ssum, \
                                             sover, n0);                                                                             \
    break;
            switch (nch) {
              CELLS_CASE(1) CELLS_CASE(2) CELLS_CASE(3) CELLS_CASE(4) CELLS_CASE(5) CELLS_CASE(6)
              CELLS_CASE(7) CELLS_CASE(8) CELLS_CASE(9) CELLS_CASE(10) CELLS_CASE(11) CELLS_CASE(12)
              default: break;
            }
#undef CELLS_CASE
          }
        } else {  // very dense: particle by particle over the windows, the row carried from window to window
          for (unsigned il = 0; il < n; ++il) {
            for (unsigned win = 0; win < ncand; win += 32u * CHMAX) {
              const bool last = win + 32u * CHMAX >= ncand;
              load_window(win, CHMAX);
              if (win == 0u) cell_tests_flush<CHMAX, true, false, false>(p, C, img, S_cell, il, il + 1u, G_cell + il, rbase_w, cut2, ltmask, lane, lhist, smax, ssum, sover, n0);
              else if (!last) cell_tests_flush<CHMAX, false, false, false>(p, C, img, S_cell, il, il + 1u, G_cell + il, rbase_w, cut2, ltmask, lane, lhist, smax, ssum, sover, n0);
              else cell_tests_flush<CHMAX, false, true, false>(p, C, img, S_cell, il, il + 1u, G_cell + il, rbase_w, cut2, ltmask, lane, lhist, smax, ssum, sover, n0);
            }
          }
        }
      } else {
        for (unsigned r0 = 0; r0 < n;) {
          if (rows_used == 32u || (r0 == 0 && rows_used + n > 32u && n <= 32u)) flush();  // keep a cell's rows together when they fit
          const unsigned take = min(n - r0, 32u - rows_used);
          if (lane >= rows_used && lane < rows_used + take) {
            my_gi = G_cell + r0 + (lane - rows_used);
            my_self = S_cell + r0 + (lane - rows_used);
            rowcnt[lane] = 0;
          }
          __syncwarp();
          for (unsigned win = 0; win < ncand; win += 32u * CHMAX) {  // one window unless the stencil holds more than 384 particles
            const unsigned nch = (min(ncand, win + 32u * CHMAX) - win + 31u) >> 5;
            load_window(win, nch);
#define CELLS_CASE(K)                                                                                                           \
  case K:                                                                                                                         \
    cell_tests<K>(p, C, img, S_cell, r0, r0 + take, rows_used, rbase_w, row_bytes, rowcnt, cut2, rowcap, ltmask, lane);              \
    break;
            switch (nch) {
              CELLS_CASE(1) CELLS_CASE(2) CELLS_CASE(3) CELLS_CASE(4) CELLS_CASE(5) CELLS_CASE(6)
              CELLS_CASE(7) CELLS_CASE(8) CELLS_CASE(9) CELLS_CASE(10) CELLS_CASE(11) CELLS_CASE(12)
              default: break;
            }
#undef CELLS_CASE
          }
          rows_used += take;
          r0 += take;
        }
      }
    }
    if (MODE == 1) flush();
  }
  // statistics of the tile: per warp into shared memory, one set of global atomics per CTA
  smax = __reduce_max_sync(0xffffffffu, smax);
  ssum = __reduce_add_sync(0xffffffffu, ssum);
  const unsigned wover = __any_sync(0xffffffffu, sover);
  if (lane == 0) {
    atomicMax(&lhist[LCAP + 1], smax);
    atomicAdd(&lhist[LCAP + 2], ssum);
    if (wover) atomicOr(&lhist[LCAP + 3], 1u);
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    Ctl* c = p.ctl;
    if (MODE == 0) {
      atomicMax(&c->max_nbr, lhist[LCAP + 1]);
      atomicAdd(&c->sum_nbr, (unsigned long long)lhist[LCAP + 2]);
    } else {
      atomicAdd(&c->sum_act, (unsigned long long)lhist[LCAP + 2]);
      if (blockIdx.x == 0) atomicAdd(&c->dens_passes, 1ull);
    }
    if (lhist[LCAP + 3]) {
      atomicOr(&c->err, ERR_OVERFLOW);
      atomicAdd(&c->overflow, 1ull);
    }
  }
  // Hand-out order of the pass that follows (MODE 0: the density pass, by decreasing list length; MODE 1: the force pass,
  // by decreasing in-range count): counting sort in shared memory, the histogram was filled on the fly.  Group g =
  // sorted particles 32 g .. 32 g + 31 (the lanes of a warp finish together); warp w takes the groups w, 2W-1-w, 2W+w,
  // ... (a long group, then a short one: the warps of a CTA finish together).  Which thread evaluates which particle
  // changes no result.
  if (threadIdx.x < 32) {  // exclusive scan of the LCAP + 1 bins by warp 0
    unsigned run = 0;
    for (unsigned b0 = 0; b0 <= LCAP; b0 += 32) {
      const unsigned k = b0 + lane;
      const unsigned c = k <= LCAP ? lhist[k] : 0u;
      unsigned incl = c;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const unsigned v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= (unsigned)o) incl += v;
      }
      if (k <= LCAP) lhist[k] = run + incl - c;
      run += __shfl_sync(0xffffffffu, incl, 31);
    }
  }
  __syncthreads();
  if (MODE == 0) {
    uint2* __restrict__ dout = p.dinfo + os;
    for (unsigned t = threadIdx.x; t < nown; t += blockDim.x) {
      const unsigned n = p.nnbr[os + t];
      dout[atomicAdd(&lhist[LCAP - min(n, LCAP)], 1u)] = make_uint2(t | ((unsigned)p.self_loc[os + t] << 16), n);
    }
  } else {
    uint2* __restrict__ fout = p.finfo + os;
    for (unsigned t = threadIdx.x; t < nown; t += blockDim.x) {
      const uint2 d = p.dinfo[os + t];
      fout[atomicAdd(&lhist[LCAP - min(d.y & 0x7FFFFFFFu, LCAP)], 1u)] = d;
    }
  }
}

__global__ void k_reset_list_stats(const DevP p, int always, int tiles) {
  if (!always && !p.ctl->rebuild) return;
  p.ctl->max_nbr = 0;
  p.ctl->sum_nbr = 0;
  if (tiles) {
    p.ctl->max_halo = 0;
    p.ctl->max_own = 0;
  }
}

// ----------------------------------------------------------------------------------------------------------------
// a5: density pass   rho_i = sum_{j != i, r < rd} 15 / (2 pi rd^3) (1 - r / rd)^2
// CTA = tile; thread = own particle; neighbours are shared-memory loads through the 16-bit list.  The same sweep
// also emits, for the force pass that follows, the compact list of the entries that are inside rc at THIS step
// (positions do not change between the two passes): the force pass then touches in-range pairs only.  The compact
// list is assembled 8 entries at a time in four registers (a 128-bit shift register that moves by 16 bits for an
// in-range entry and by 0 otherwise: no branch) and stored as 16-byte chunks.
// ----------------------------------------------------------------------------------------------------------------
template <bool HAS_WALL>
__device__ __forceinline__ void density_entry(const DevP& p, const unsigned pbase, const float4 xi, const unsigned walli,
                                              const unsigned j, float& rho, unsigned& a0, unsigned& a1, unsigned& a2,
                                              unsigned& a3, unsigned& na, uint4*& ao) {
  MDPD_CHECK(p, j <= p.tile_cap);
  const float4 xj = lds4(pbase + (j << 4));  // padding entries hit the far-away sentinel
  const float dx = xi.x - xj.x, dy = xi.y - xj.y, dz = xi.z - xj.z;
  const float r2 = dx * dx + dy * dy + dz * dz;
  // The logic pipe (min/max, compares, shifts, selects) issues at half the rate of the FP32 pipe and bounds this loop:
  // the clamps are saturate modifiers of the FMAs, the two-sided range test is one add and one unsigned compare.
  const float w = __saturatef(fmaf(-sqrt_fast(r2), p.inv_rd, 1.0f));  // 0 beyond rd; 1 at r = 0 (coincident particles, R10)
  rho = fmaf(w, w, rho);
  // 1e-12 < r2 < rc2 (R10): r2 - 1e-12 is negative below the lower bound (huge as an unsigned), and equals r2 wherever
  // the upper bound could matter (1e-12 is far below half an ulp of rc2)
  bool in = f2u(r2 - 1e-12f) < f2u(p.rc2 - 1e-12f);  // interacts at this step
  if (HAS_WALL) in = in && !(walli & (f2u(xj.w) >> 31));  // frozen-frozen pairs do not (R8)
  const unsigned sh = in ? 16u : 0u;
  a0 = __funnelshift_r(a0, a1, sh);
  a1 = __funnelshift_r(a1, a2, sh);
  a2 = __funnelshift_r(a2, a3, sh);
  a3 = __funnelshift_r(a3, j, sh);
  na += sh >> 4;
  if (in && (na & 7u) == 0u) {
    *ao = make_uint4(a0, a1, a2, a3);
    ao += p.N;
  }
}

constexpr int PRE = 2;  // rounds whose hand-out record and first list chunk are requested before the tile is staged

// TPB: most threads per CTA.  A tile is handed out in two rounds of one particle per thread; 384 threads (three resident
// CTAs at 56 registers) cover 768 own particles, tiles that hold more (cell edge above 1.255 at number density 6) get
// the 416-thread instantiation (48 registers, a few spills) instead of a third, almost empty round: 3.38 -> 3.14 ms per
// launch on config 4a at skin 0.27 (profiles/r2_final.md).
template <bool HAS_WALL, bool ALL, int TPB>
__global__ void __launch_bounds__(TPB, DENS_MINB) k_density(const DevP p) {
  extern __shared__ __align__(16) unsigned char smraw[];
  const TileSmem sm = carve_smem(smraw, p.tile_cap, false);
  const unsigned cur = p.ctl->cur;
  const TileInfo T = p.tiles[blockIdx.x];
  const uint4 hdr = p.runs[(size_t)blockIdx.x * p.run_stride];
  const unsigned ahead = p.sms * DENS_MINB;
  const uint4 R0 = first_record(p, ahead);
  const uint4 hdrn = p.runs[(size_t)min(blockIdx.x + ahead, gridDim.x - 1u) * p.run_stride];
  const unsigned os = hdr.w, nown = hdr.z >> 16;
  const unsigned warp = threadIdx.x >> 5, lane = threadIdx.x & 31, W = blockDim.x >> 5;
  const unsigned ngroups = (nown + 31u) >> 5;
  // the first rounds' records and list heads are in flight while the tile is staged
  uint2 info[PRE];
  uint4 head[PRE];
#pragma unroll
  for (int r = 0; r < PRE; ++r) {
    const unsigned g = group_of_round(r, warp, W), t = g * 32u + lane;
    info[r] = (g < ngroups && t < nown) ? p.dinfo[os + t] : make_uint2(0u, 0u);
  }
#pragma unroll
  for (int r = 0; r < PRE; ++r) head[r] = info[r].y ? p.nbr[os + (info[r].x & 0xFFFFu)] : make_uint4(0, 0, 0, 0);
  if (!((p.tma_staging & 1u) ? stage_bulk<false>(p, T, hdr, R0, p.pos[cur], nullptr, sm) : stage_fast<false>(p, T, hdr, R0, p.pos[cur], nullptr, sm)))
    return;  // flagged by k_tile_recipe
  prefetch_handout(p, ahead, hdrn, p.dinfo, p.nbr);
  float4* __restrict__ vel = p.vel[cur];
  const unsigned sent = p.tile_cap;
  const unsigned pbase = smem_addr(sm.spos);
  unsigned* const hist = sm.hbase;  // [LCAP + 1] bins of the sort below (bin 0 = longest) + the in-range pair count; the
                                    // shift table that lived here is dead after staging
  for (unsigned k = threadIdx.x; k < HTAB; k += blockDim.x) hist[k] = 0u;
  unsigned na_sum = 0;
  uint2 frec[PRE];  // this thread's records for the force pass: x as in dinfo, y = in-range count (bit 31: frozen, skip)
#pragma unroll
  for (int r = 0; r < PRE; ++r) frec[r] = make_uint2(0u, 0u);
  for (unsigned r = 0; r * W < ngroups; ++r) {
    const unsigned g = group_of_round(r, warp, W);
    const unsigned t = g * 32u + lane;
    if (g >= ngroups || t >= nown) continue;
    uint2 rec;
    uint4 nxt;
    if (r < PRE) {
      rec = r == 0 ? info[0] : info[PRE - 1];
      nxt = r == 0 ? head[0] : head[PRE - 1];
    } else {
      rec = p.dinfo[os + t];
      nxt = rec.y ? p.nbr[os + (rec.x & 0xFFFFu)] : make_uint4(0, 0, 0, 0);
    }
    const unsigned i = os + (rec.x & 0xFFFFu);
    MDPD_CHECK(p, i < p.N && (rec.x & 0xFFFFu) < nown && (rec.x >> 16) < p.tile_cap && rec.y <= p.cap);
    const float4 xi = sm.spos[rec.x >> 16];
    const unsigned walli = f2u(xi.w) >> 31;
    const unsigned nn = rec.y;
    const uint4* __restrict__ lst = p.nbr + i;
    uint4* ao = p.act + i;  // next chunk to write
    float rho = 0.0f;
    unsigned a0 = 0, a1 = 0, a2 = 0, a3 = 0, na = 0;
    for (unsigned k0 = 0; k0 < nn; k0 += 8) {
      const uint4 e = nxt;
      if (k0 + 8 < nn) nxt = lst[(size_t)((k0 >> 3) + 1) * p.N];  // next chunk in flight while this one is evaluated
      density_entry<HAS_WALL>(p, pbase, xi, walli, e.x & 0xFFFFu, rho, a0, a1, a2, a3, na, ao);
      density_entry<HAS_WALL>(p, pbase, xi, walli, e.x >> 16, rho, a0, a1, a2, a3, na, ao);
      density_entry<HAS_WALL>(p, pbase, xi, walli, e.y & 0xFFFFu, rho, a0, a1, a2, a3, na, ao);
      density_entry<HAS_WALL>(p, pbase, xi, walli, e.y >> 16, rho, a0, a1, a2, a3, na, ao);
      density_entry<HAS_WALL>(p, pbase, xi, walli, e.z & 0xFFFFu, rho, a0, a1, a2, a3, na, ao);
      density_entry<HAS_WALL>(p, pbase, xi, walli, e.z >> 16, rho, a0, a1, a2, a3, na, ao);
      density_entry<HAS_WALL>(p, pbase, xi, walli, e.w & 0xFFFFu, rho, a0, a1, a2, a3, na, ao);
      density_entry<HAS_WALL>(p, pbase, xi, walli, e.w >> 16, rho, a0, a1, a2, a3, na, ao);
    }
    if (na & 7u) {  // last, partial chunk: pad with the sentinel
      for (unsigned q = na & 7u; q < 8u; ++q) {
        a0 = __funnelshift_r(a0, a1, 16);
        a1 = __funnelshift_r(a1, a2, 16);
        a2 = __funnelshift_r(a2, a3, 16);
        a3 = __funnelshift_r(a3, sent, 16);
      }
      *ao = make_uint4(a0, a1, a2, a3);
    }
    p.nact[i] = (unsigned short)na;
    na_sum += na;
    vel[i].w = rho * p.Krho;
    const unsigned fy = (HAS_WALL && !ALL && walli) ? 0x80000000u : na;  // frozen: force not needed (R8)
    if (r == 0) frec[0] = make_uint2(rec.x, fy);
    else if (r < PRE) frec[PRE - 1] = make_uint2(rec.x, fy);
  }
  // Hand-out records of the force pass that follows: own particles by decreasing in-range count of this step (counting
  // sort; the keys of the first PRE rounds are still in registers).  The in-range pair count of the tile (the force
  // pass's algorithmic work, a statistic) rides on the same barriers.
  auto round_record = [&](unsigned r, uint2& out) {
    const unsigned g = group_of_round(r, warp, W), t = g * 32u + lane;
    if (g >= ngroups || t >= nown) return false;
    if (r == 0) out = frec[0];
    else if (r < PRE) out = frec[PRE - 1];
    else {
      const uint2 d = p.dinfo[os + t];
      const bool skip = HAS_WALL && !ALL && (f2u(sm.spos[d.x >> 16].w) >> 31);
      out = make_uint2(d.x, skip ? 0x80000000u : (unsigned)p.nact[os + (d.x & 0xFFFFu)]);
    }
    return true;
  };
  na_sum = __reduce_add_sync(0xffffffffu, na_sum);
  __syncthreads();  // hist is zero, every particle of the tile is done
  if (lane == 0 && na_sum) atomicAdd(&hist[HTAB - 1], na_sum);
  for (unsigned r = 0; r * W < ngroups; ++r) {
    uint2 fr;
    if (round_record(r, fr)) atomicAdd(&hist[LCAP - min(fr.y & 0x7FFFFFFFu, LCAP)], 1u);
  }
  __syncthreads();
  if (threadIdx.x < 32) {  // exclusive scan of the LCAP + 1 bins by warp 0
    unsigned run = 0;
    for (unsigned b0 = 0; b0 <= LCAP; b0 += 32) {
      const unsigned k = b0 + lane;
      const unsigned c = k <= LCAP ? hist[k] : 0u;
      unsigned incl = c;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const unsigned v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
      }
      if (k <= LCAP) hist[k] = run + incl - c;
      run += __shfl_sync(0xffffffffu, incl, 31);
    }
    if (lane == 0) {
      atomicAdd(&p.ctl->sum_act, (unsigned long long)hist[HTAB - 1]);
      if (blockIdx.x == 0) atomicAdd(&p.ctl->dens_passes, 1ull);
    }
  }
  __syncthreads();
  uint2* __restrict__ fout = p.finfo + os;
  for (unsigned r = 0; r * W < ngroups; ++r) {
    uint2 fr;
    if (round_record(r, fr)) fout[atomicAdd(&hist[LCAP - min(fr.y & 0x7FFFFFFFu, LCAP)], 1u)] = fr;
  }
}

// ----------------------------------------------------------------------------------------------------------------
// a6: pair-force pass (Eq. (1); L186 body force)
//   F_ij = [A wC + B (rho_i + rho_j) wd - gamma wC^2 (e.v_ij) + sigma wC xi_ij / sqrt(dt)] e_ij ,  s = 1
// Full list: every pair is evaluated from both ends; the symmetric hash makes F_ij = -F_ji bitwise.
// Walks the compact in-range list the density pass wrote for this step: every evaluated pair interacts.  The loop body
// has no branch: the padding of a particle's last chunk points at the far-away sentinel slot, whose weights clamp to 0.
// ----------------------------------------------------------------------------------------------------------------
struct ForceAcc {
  float x, y, z;
};

// MULTI: per-type-pair (A, B, gamma, sig_c) from the table `ab` in shared memory (row = species of i), else the handle's
// VIRIAL: also accumulate r_a F^C_b of the pair (conservative part of the stress, section 4.1 of the paper) into vir[6]
template <bool MULTI, bool VIRIAL, bool SPOW>
__device__ __forceinline__ void force_entry(const DevP& p, const unsigned pbase, const unsigned vbase, const float4 xi,
                                            const float4 vi, const unsigned tagi, const unsigned j, const HashKeys& K,
                                            const float4* ab, ForceAcc& acc, float* vir) {
  MDPD_CHECK(p, j <= p.tile_cap);
  const float4 xj = lds4(pbase + (j << 4));
  const float4 vj = lds4(vbase + (j << 4));
  const float dx = xi.x - xj.x, dy = xi.y - xj.y, dz = xi.z - xj.z;
  const float r2 = dx * dx + dy * dy + dz * dz;  // > 1e-12 for list entries; 3e18 for the sentinel
  const float rinv = rsqrt_fast(r2);
  const float r = r2 * rinv;
  const float w = __saturatef(fmaf(-r, p.inv_rc, 1.0f));  // > 0 for in-range entries, 0 for the sentinel
  float Aij = p.A, Bij = p.B, gam = p.gamma, sigc = p.sig_c;
  if (MULTI) {  // the species sits in bits 28..30 of the particle word (A_SL, B_SL; L75: gamma, sigma)
    const float4 t = ab[(f2u(xj.w) >> TAG_BITS) & (MAXTYPES - 1u)];
    Aij = t.x;
    Bij = t.y;
    gam = t.z;
    sigc = t.w;
  }
  float F = Aij * w;
  const float wd = __saturatef(fmaf(-r, p.inv_rd, 1.0f));
  F += Bij * (vi.w + vj.w) * wd;
  if (VIRIAL) {  // F is the conservative force here; the sentinel contributes 0 * finite
    const float c = F * rinv;
    vir[0] += c * dx * dx;
    vir[1] += c * dy * dy;
    vir[2] += c * dz * dz;
    vir[3] += c * dx * dy;
    vir[4] += c * dx * dz;
    vir[5] += c * dy * dz;
  }
  const float ev = (dx * (vi.x - vj.x) + dy * (vi.y - vj.y) + dz * (vi.z - vj.z)) * rinv;
  // wR = w^s (wD = wR^2); s = 1 unless SPOW.  w = 0 (sentinel) gives exp2(-inf) = 0.
  const float wR = SPOW ? __powf(w, p.s_exp) : w;
  F -= gam * wR * wR * ev;
  const unsigned h = pair_hash(tagi, f2u(xj.w) & TAG_MASK, K);
  const float xi_s = (float)((int)(h >> 8) - (1 << 23));  // exact
  F += sigc * wR * xi_s;
  const float Fr = F * rinv;
  acc.x += Fr * dx;
  acc.y += Fr * dy;
  acc.z += Fr * dz;
}

template <bool ALL, bool MULTI, bool VIRIAL = false, bool SPOW = false>  // SPOW: general exponent s of wR; ALL: also evaluate the (never used) forces on frozen particles, for parity checks
__global__ void __launch_bounds__(TILE_TPB, MINB) k_force(const DevP p) {
  extern __shared__ __align__(16) unsigned char smraw[];
  __shared__ float4 s_ab[MULTI ? MAXTYPES * MAXTYPES : 1];
  if (MULTI) {
    for (unsigned q = threadIdx.x; q < MAXTYPES * MAXTYPES; q += blockDim.x)  // ordered by stage_fast's barriers
      s_ab[q] = make_float4(p.AB[q].x, p.AB[q].y, p.GS[q].x, p.GS[q].y);
  }
  const TileSmem sm = carve_smem(smraw, p.tile_cap, true);
  const unsigned cur = p.ctl->cur;
  const TileInfo T = p.tiles[blockIdx.x];
  const uint4 hdr = p.runs[(size_t)blockIdx.x * p.run_stride];
  const unsigned ahead = p.sms * MINB;
  const uint4 R0 = first_record(p, ahead);
  const uint4 hdrn = p.runs[(size_t)min(blockIdx.x + ahead, gridDim.x - 1u) * p.run_stride];
  const unsigned os = hdr.w, nown = hdr.z >> 16;
  const unsigned warp = threadIdx.x >> 5, lane = threadIdx.x & 31, W = blockDim.x >> 5;
  const unsigned ngroups = (nown + 31u) >> 5;
  const unsigned sentw = p.tile_cap | (p.tile_cap << 16);
  // the first rounds' records (written by the density pass of this step) and list heads are in flight while the
  // tile is staged
  uint2 info[PRE];
  uint4 head[PRE];
#pragma unroll
  for (int r = 0; r < PRE; ++r) {
    const unsigned g = group_of_round(r, warp, W), t = g * 32u + lane;
    info[r] = (g < ngroups && t < nown) ? p.finfo[os + t] : make_uint2(0u, 0x80000000u);
  }
#pragma unroll
  for (int r = 0; r < PRE; ++r)
    head[r] = (info[r].y & 0x7FFFFFFFu) ? p.act[os + (info[r].x & 0xFFFFu)] : make_uint4(sentw, sentw, sentw, sentw);
  if (!((p.tma_staging & 2u) ? stage_bulk<true>(p, T, hdr, R0, p.pos[cur], p.vel[cur], sm) : stage_fast<true>(p, T, hdr, R0, p.pos[cur], p.vel[cur], sm)))
    return;
  prefetch_handout(p, ahead, hdrn, p.finfo, p.act);
  HashKeys K = make_keys(p.ctl->step, p.seed);
#pragma unroll
  for (int q = 0; q < 6; ++q) K.k[q] = pin(K.k[q]);
  const unsigned pbase = smem_addr(sm.spos), vbase = smem_addr(sm.svel);
  double vsum[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
  for (unsigned r = 0; r * W < ngroups; ++r) {
    const unsigned g = group_of_round(r, warp, W);
    const unsigned t = g * 32u + lane;
    if (g >= ngroups || t >= nown) continue;
    uint2 rec;
    uint4 nxt;
    if (r < PRE) {
      rec = r == 0 ? info[0] : info[PRE - 1];
      nxt = r == 0 ? head[0] : head[PRE - 1];
    } else {
      rec = p.finfo[os + t];
      nxt = (rec.y & 0x7FFFFFFFu) ? p.act[os + (rec.x & 0xFFFFu)] : make_uint4(sentw, sentw, sentw, sentw);
    }
    const unsigned i = os + (rec.x & 0xFFFFu);
    if (rec.y >> 31) {  // frozen particles are never integrated (R8): their force is not needed; reported as zero
      p.force[i] = make_float4(0.f, 0.f, 0.f, 0.f);
      continue;
    }
    const unsigned li = rec.x >> 16;
    MDPD_CHECK(p, i < p.N && (rec.x & 0xFFFFu) < nown && li < p.tile_cap && rec.y <= p.cap);
    const float4 xi = sm.spos[li];
    const unsigned wi = f2u(xi.w);
    const unsigned tagi = wi & TAG_MASK;
    const float4* const ab = s_ab + (MULTI ? ((wi >> TAG_BITS) & (MAXTYPES - 1u)) * MAXTYPES : 0u);
    const float4 vi = sm.svel[li];
    const unsigned na = rec.y;
    ForceAcc acc = {0.f, 0.f, 0.f};
    float vir[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    const uint4* __restrict__ lst = p.act + i;
    for (unsigned k0 = 0; k0 < na; k0 += 8) {
      const uint4 e = nxt;
      if (k0 + 8 < na) nxt = lst[(size_t)((k0 >> 3) + 1) * p.N];  // next chunk in flight
      force_entry<MULTI, VIRIAL, SPOW>(p, pbase, vbase, xi, vi, tagi, e.x & 0xFFFFu, K, ab, acc, vir);
      force_entry<MULTI, VIRIAL, SPOW>(p, pbase, vbase, xi, vi, tagi, e.x >> 16, K, ab, acc, vir);
      force_entry<MULTI, VIRIAL, SPOW>(p, pbase, vbase, xi, vi, tagi, e.y & 0xFFFFu, K, ab, acc, vir);
      force_entry<MULTI, VIRIAL, SPOW>(p, pbase, vbase, xi, vi, tagi, e.y >> 16, K, ab, acc, vir);
      if (k0 + 4 < na) {  // the second half of the chunk holds at least one entry
        force_entry<MULTI, VIRIAL, SPOW>(p, pbase, vbase, xi, vi, tagi, e.z & 0xFFFFu, K, ab, acc, vir);
        force_entry<MULTI, VIRIAL, SPOW>(p, pbase, vbase, xi, vi, tagi, e.z >> 16, K, ab, acc, vir);
        force_entry<MULTI, VIRIAL, SPOW>(p, pbase, vbase, xi, vi, tagi, e.w & 0xFFFFu, K, ab, acc, vir);
        force_entry<MULTI, VIRIAL, SPOW>(p, pbase, vbase, xi, vi, tagi, e.w >> 16, K, ab, acc, vir);
      }
    }
    if (!(wi >> 31)) {
      acc.x += p.fgx;
      acc.y += p.fgy;
      acc.z += p.fgz;
    }
    p.force[i] = make_float4(acc.x, acc.y, acc.z, 0.0f);
    if (VIRIAL) {
#pragma unroll
      for (int q = 0; q < 6; ++q) vsum[q] += (double)vir[q];
    }
  }
  if (VIRIAL) {  // all lanes of the warp arrive here (the round loop has no early return)
#pragma unroll
    for (int q = 0; q < 6; ++q) {
      double v = vsum[q];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
      if (lane == 0 && v != 0.0) atomicAdd(&p.ctl->vir[q], v);
    }
  }
}

// ----------------------------------------------------------------------------------------------------------------
// parity exports
// ----------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(512) k_pairs(const DevP p, float rcut2, uint2* out, unsigned long long cap,
                                               unsigned long long* count) {
  extern __shared__ __align__(16) unsigned char smraw[];
  const TileSmem sm = carve_smem(smraw, p.tile_cap, false);
  const unsigned cur = p.ctl->cur;
  const TileInfo T = p.tiles[blockIdx.x];
  if (stage_tile<false>(p, T, p.pos[cur], nullptr, sm) == 0xFFFFFFFFu) return;
  const unsigned os = p.cell_start[T.rank0], oe = p.cell_start[T.rank0 + T.ncell_own];
  for (unsigned i = os + threadIdx.x; i < oe; i += blockDim.x) {
    const float4 xi = sm.spos[p.self_loc[i]];
    const unsigned tagi = f2u(xi.w) & TAG_MASK;
    const unsigned n = p.nnbr[i];
    {
      const uint4* lst = p.nbr + i;
      for (unsigned k = 0; k < n; ++k) {
        const uint4 e = lst[(size_t)(k >> 3) * p.N];
        const unsigned w = (k & 4) ? ((k & 2) ? e.w : e.z) : ((k & 2) ? e.y : e.x);
        const float4 xj = sm.spos[(k & 1) ? (w >> 16) : (w & 0xFFFFu)];
        const unsigned tagj = f2u(xj.w) & TAG_MASK;
        if (tagi >= tagj) continue;
        const float dx = xi.x - xj.x, dy = xi.y - xj.y, dz = xi.z - xj.z;
        const float r2 = dx * dx + dy * dy + dz * dz;
        if (r2 < rcut2) {
          unsigned long long s = atomicAdd(count, 1ull);
          if (s < cap) out[s] = make_uint2(tagi, tagj);
        }
      }
    }
  }
}

}  // namespace (left for a moment: the scratch array below sits at file scope)

// ----------------------------------------------------------------------------------------------------------------
// Fixed scratch of mdpd_get_pairs_static: the hit counter of k_pairs (first 8 bytes; the rest of the first 256 bytes
// is padding that keeps the pair buffer aligned) followed by room for MDPD_STATIC_PAIRS_MAX (tag, tag) pairs.  It is
// part of the library image, so every GPU that loads the library carries these ~4 MiB until the process exits, and
// nobody ever has to allocate or free them.
//
// The name below is only usable as an address inside device code.  On the host it is a stand-in symbol of the
// runtime, NOT a device pointer: a kernel handed `g_pairs_scratch` from host code would fault (or, where the GPU can
// reach host memory, scribble over whatever lives there).  Host code therefore asks the runtime for the real
// address, once per device and with that device current (static_pairs_scratch below), and hands THAT to the kernel.
// ----------------------------------------------------------------------------------------------------------------
constexpr size_t STATIC_PAIRS_HEAD = 256;  // bytes in front of the pair buffer (counter + padding)
static __device__ __align__(256) unsigned char g_pairs_scratch[STATIC_PAIRS_HEAD + (size_t)MDPD_STATIC_PAIRS_MAX * sizeof(uint2)];

constexpr int STATIC_MAXDEV = 64;                    // device ordinals this table covers
static unsigned char* g_pairs_scratch_addr[STATIC_MAXDEV];  // resolved device address per ordinal, nullptr = not yet asked
static std::mutex g_pairs_scratch_mu;

// Device address of g_pairs_scratch on `device`, which must be the current device.  The first call per device asks
// the runtime (this is what makes the first mdpd_get_pairs_static call on a device a set-up call); later calls read
// the table.  Returns cudaSuccess or the runtime's error.
static cudaError_t static_pairs_scratch(int device, unsigned char** out) {
  if (device < 0 || device >= STATIC_MAXDEV) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_pairs_scratch_mu);
  if (!g_pairs_scratch_addr[device]) {
    void* ptr = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&ptr, g_pairs_scratch);
    if (e != cudaSuccess) return e;
    if (!ptr) return cudaErrorInvalidSymbol;
    g_pairs_scratch_addr[device] = (unsigned char*)ptr;
  }
  *out = g_pairs_scratch_addr[device];
  return cudaSuccess;
}

namespace {

__global__ void k_rng_fill(unsigned long long n, const uint2* __restrict__ pairs, unsigned step, unsigned seed,
                           unsigned* __restrict__ out) {
  unsigned long long q = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= n) return;
  const HashKeys K = make_keys(step, seed);
  out[q] = pair_hash(pairs[q].x, pairs[q].y, K);
}

// ----------------------------------------------------------------------------------------------------------------
// Issue-rate probe (mdpd_probe_issue_rates): register-only kernels, 8 independent chains per thread, so that the pipe
// and not the dependency latency bounds them.  KIND 0: FFMA; 1: LOP3 + VIMNMX (the logic pipe); 2: IMAD.WIDE + the
// add that closes its chain.  The unused result is stored under a condition that never holds.
// ----------------------------------------------------------------------------------------------------------------
constexpr int PROBE_CH = 8, PROBE_ITER = 2048, PROBE_TPB = 1024;
template <int KIND>
__global__ void __launch_bounds__(PROBE_TPB) k_probe(float* out, float a, float b, unsigned ua, unsigned ub) {
  float x[PROBE_CH];
  unsigned u[PROBE_CH];
  unsigned long long w[PROBE_CH];
#pragma unroll
  for (int c = 0; c < PROBE_CH; ++c) {
    x[c] = (float)threadIdx.x * 1e-3f + (float)c;
    u[c] = threadIdx.x * 77u + (unsigned)c;
    w[c] = u[c];
  }
  for (int it = 0; it < PROBE_ITER; ++it) {
#pragma unroll
    for (int c = 0; c < PROBE_CH; ++c) {
      if (KIND == 0) x[c] = fmaf(x[c], a, b);
      if (KIND == 1) u[c] = max(u[c], ua) ^ ub;
      if (KIND == 2) w[c] = (unsigned long long)(unsigned)w[c] * 0xD256D193ull + (w[c] >> 32);
    }
  }
  float sum = 0.f;
#pragma unroll
  for (int c = 0; c < PROBE_CH; ++c) sum += x[c] + (float)u[c] + (float)w[c];
  if (sum == 12345.678f) out[0] = sum;
}

// ----------------------------------------------------------------------------------------------------------------
// host side
// ----------------------------------------------------------------------------------------------------------------
inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

struct Layout {
  size_t pos[2], vel[2], force, xbuild, cell_rank, cell_count, cell_start, scan_bsum, pcell, order, nbr,
      act, nact, nnbr, self_loc, tiles, runs, dperm, fperm, mask, ctl, stage, total;
  unsigned ncx, ncy, ncz, ncell, cap, cap_act, scan_blocks;
  float rlist;
};

bool make_layout(const mdpd_params& p, uint64_t n, int has_mask, const uint32_t* md, Layout& L, std::string* why) {
  auto fail = [&](const char* m) {
    if (why) *why = m;
    return false;
  };
  if (!(p.rc > 0) || !(p.rd > 0) || !(p.rd <= p.rc)) return fail("need 0 < rd <= rc");
  if (!(p.skin >= 0)) return fail("skin must be >= 0");
  if (!(p.dt > 0) || !(p.mass > 0)) return fail("dt and mass must be > 0");
  if (!(p.s > 0.0f) || p.s > 4.0f) return fail("the exponent s of wR = (1 - r/rc)^s must be in (0, 4] (DESIGN.md R15)");
  if (p.reorder_every > 1) return fail("reorder_every is reserved and must be 0 or 1: the counting sort into tiles IS the reorder, at every rebuild (DESIGN.md R16)");
  if (n >= (1ull << TAG_BITS)) return fail("n must be < 2^28");
  L.rlist = p.rc + p.skin;
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
  const double m_list = 4.0 / 3.0 * PI * std::pow((double)L.rlist, 3) * dens;
  if (p.max_neigh == 0) L.cap = std::min<unsigned>(LCAP, (unsigned)(std::ceil((m_list + 6.0 * std::sqrt(m_list) + 8.0) / 8.0) * 8.0));
  else L.cap = (p.max_neigh + 7u) / 8u * 8u;
  if (L.cap > LCAP) return fail("max_neigh must be <= 128 (the list build assembles a particle's list in shared memory)");
  {  // capacity of the per-step in-range (r < rc) lists of the list-free path
    const double m_act = 4.0 / 3.0 * PI * std::pow((double)p.rc, 3) * dens;
    L.cap_act = std::min<unsigned>(L.cap, (unsigned)(std::ceil((m_act + 6.0 * std::sqrt(m_act) + 8.0) / 8.0) * 8.0));
  }
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
  L.nbr = take(N * 2 * L.cap);
  L.act = take(N * 2 * L.cap);
  L.nact = take(N * 2);
  L.nnbr = take(N * 4);
  L.self_loc = take(N * 2);
  L.tiles = take((size_t)L.ncell * sizeof(TileInfo));  // worst case: one cell per tile
  L.runs = take(((size_t)L.ncell * 32 + 4096) * 16);   // worst case: one cell per tile: header + 27 records + 4 (slot table)
  L.dperm = take(N * 8);
  L.fperm = take(N * 8);
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
  bool has_wall = false;  // some particle is frozen (type 1)
  unsigned ntypes = 0, frozen_mask = 0;        // mdpd_set_pair_params
  float pairA[MAXTYPES * MAXTYPES] = {}, pairB[MAXTYPES * MAXTYPES] = {};
  bool have_gs = false;                        // mdpd_set_pair_gamma_sigma
  float pairG[MAXTYPES * MAXTYPES] = {}, pairS[MAXTYPES * MAXTYPES] = {};
  uint64_t launches = 0;         // kernels launched directly (graph replays are added from graph_steps / ctl)
  uint64_t host_step = 0;
  cudaStream_t ls = nullptr;     // stream the LAUNCH macro targets (the handle's stream, or the capture stream)
  cudaStream_t cap_stream = nullptr;
  cudaGraph_t graph = nullptr;   // one timestep: integrate -> IF(trigger){sort + list build} -> density -> force
  cudaGraphExec_t graph_exec = nullptr;
  cudaGraphConditionalHandle cond = 0;
  bool graph_dirty = true;       // kernel arguments (DevP) changed since the capture
  bool use_graph = true;
  bool pending_B = false;        // the second half kick of the last step has not been applied yet
  uint64_t graph_steps = 0;
  int tile_dim[3] = {4, 4, 4};
  unsigned block = 256;          // threads per CTA of the force pass
  unsigned block_dens = 256;     // threads per CTA of the density pass
  unsigned blocks_from = 0;      // the tile occupancy (max_own) the two block sizes were chosen for
  unsigned cells_warps[2] = {4, 4};  // warps per CTA of k_cells (list build / list-free pass)
  size_t smem_cells[2] = {0, 0};
  bool direct = false;           // MDPD_FLAG_DIRECT: no Verlet list, neighbours straight from the cells every step
  unsigned chain_launches = 9;   // kernels of the rebuild chain
  size_t smem_pos = 0, smem_posvel = 0;
  size_t smem_limit = 0;         // cudaDevAttrMaxSharedMemoryPerBlockOptin
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

enum ProfSlot { PS_INTEGRATE = 0, PS_CELL_COUNT, PS_SCAN, PS_CELL_FILL, PS_PERMUTE, PS_RECIPE, PS_CELLS_LIST, PS_CELLS_DIRECT,
                PS_DENSITY, PS_FORCE, PS_OTHER, PS_COUNT };
const char* const kProfNames[PS_COUNT] = {"k_integrate", "k_cell_count", "k_scan", "k_cell_fill", "k_permute", "k_tile_recipe",
                                          "k_cells_list", "k_cells_direct", "k_density", "k_force", "other"};

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
  d.nbr = (uint4*)(w + L.nbr);
  d.act = (uint4*)(w + L.act);
  d.nact = (unsigned short*)(w + L.nact);
  d.nnbr = (unsigned*)(w + L.nnbr);
  d.self_loc = (unsigned short*)(w + L.self_loc);
  d.tiles = (const TileInfo*)(w + L.tiles);
  d.runs = (uint4*)(w + L.runs);
  d.dinfo = (uint2*)(w + L.dperm);
  d.finfo = (uint2*)(w + L.fperm);
  d.mask = (const unsigned char*)(w + L.mask);
  d.ctl = (Ctl*)(w + L.ctl);
  d.N = (unsigned)h->n;
  d.ncell = L.ncell;
  d.cap = L.cap;
  d.ncx = L.ncx; d.ncy = L.ncy; d.ncz = L.ncz;
  d.Lx = p.box[0]; d.Ly = p.box[1]; d.Lz = p.box[2];
  d.icx = (float)((double)L.ncx / (double)p.box[0]);
  d.icy = (float)((double)L.ncy / (double)p.box[1]);
  d.icz = (float)((double)L.ncz / (double)p.box[2]);
  d.rlist2 = L.rlist * L.rlist;
  d.edge_x = (float)((double)p.box[0] / (double)L.ncx);
  d.edge_y = (float)((double)p.box[1] / (double)L.ncy);
  d.edge_z = (float)((double)p.box[2] / (double)L.ncz);
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
  d.s_exp = p.s;
  d.ntypes = h->ntypes;
  d.frozen_mask = h->frozen_mask;
  for (unsigned a = 0; a < MAXTYPES; ++a)
    for (unsigned b = 0; b < MAXTYPES; ++b) {
      const bool in = a < h->ntypes && b < h->ntypes;
      d.AB[a * MAXTYPES + b] = make_float2(in ? h->pairA[a * h->ntypes + b] : p.A, in ? h->pairB[a * h->ntypes + b] : p.B);
      const bool gs = in && h->have_gs;
      const double sg = gs ? (double)h->pairS[a * h->ntypes + b] : (double)p.sigma;
      d.GS[a * MAXTYPES + b] = make_float2(gs ? h->pairG[a * h->ntypes + b] : p.gamma,
                                           (float)(sg * std::sqrt(3.0) * std::ldexp(1.0, -23) / std::sqrt((double)p.dt)));
    }
}

// Sort order of the cells: tiles of tdim[0] x tdim[1] x tdim[2] cells enumerated along the Z-curve (Morton order of
// the tile coordinates: neighbouring tiles are close in memory and in L2), cells x-fastest inside a tile (the cells
// of a tile row, and the whole tile, are contiguous runs of particles).
void build_tile_ranks(const Layout& L, const int tdim[3], std::vector<unsigned>& rank, std::vector<TileInfo>& tiles) {
  rank.assign(L.ncell, 0u);
  tiles.clear();
  const unsigned ntx = (L.ncx + tdim[0] - 1) / tdim[0], nty = (L.ncy + tdim[1] - 1) / tdim[1],
                 ntz = (L.ncz + tdim[2] - 1) / tdim[2];
  unsigned mx = std::max(ntx, std::max(nty, ntz));
  int bits = 0;
  while ((1u << bits) < mx) ++bits;
  auto compact = [](unsigned long long v) {  // every third bit
    unsigned r = 0;
    for (int b = 0; b < 11; ++b) r |= (unsigned)((v >> (3 * b)) & 1ull) << b;
    return r;
  };
  unsigned next = 0;
  const unsigned long long ncodes = 1ull << (3 * bits);
  for (unsigned long long code = 0; code < ncodes; ++code) {
    const unsigned tx = compact(code), ty = compact(code >> 1), tz = compact(code >> 2);
    if (tx >= ntx || ty >= nty || tz >= ntz) continue;
    // tile t of nt along a dimension of nc cells starts at floor(t nc / nt): extents differ by at most one cell, no thin
    // remainder tile at the upper faces (137 cells: 32 tiles of 4 and 3 of 3 instead of 34 of 4 and one of 1)
    auto start = [](unsigned t, unsigned nt, unsigned nc) { return (int)((unsigned long long)t * nc / nt); };
    TileInfo T;
    T.c0x = start(tx, ntx, L.ncx); T.c0y = start(ty, nty, L.ncy); T.c0z = start(tz, ntz, L.ncz);
    T.ex = start(tx + 1, ntx, L.ncx) - T.c0x;
    T.ey = start(ty + 1, nty, L.ncy) - T.c0y;
    T.ez = start(tz + 1, ntz, L.ncz) - T.c0z;
    T.rank0 = next;
    T.ncell_own = (unsigned)(T.ex * T.ey * T.ez);
    for (int lz = 0; lz < T.ez; ++lz)
      for (int ly = 0; ly < T.ey; ++ly)
        for (int lx = 0; lx < T.ex; ++lx)
          rank[((size_t)(T.c0z + lz) * L.ncy + (T.c0y + ly)) * L.ncx + (T.c0x + lx)] = next++;
    tiles.push_back(T);
  }
}

// Threads per CTA of the density / force passes: the own particles of a tile are handed out in two rounds of one
// particle per thread (every warp gets a long and a short group, see k_cells' tail), so a CTA wants half the fullest
// tile's population.  The density pass has two instantiations (384 threads at 56 registers, 416 at 48): the wider one
// only when the fullest tile exceeds what 384 threads cover by more than 5 % (a third, almost empty round in a few tiles
// costs less than the spills).  Re-evaluated by mdpd_step from the occupancy the last synchronising call saw.
bool choose_blocks(mdpd_ctx* h, unsigned max_own) {
  const unsigned half_own = ((max_own + 1u) / 2u + 31u) / 32u * 32u;
  const unsigned b = std::min<unsigned>(TILE_TPB, std::max(64u, half_own));
  const unsigned bd = (double)max_own > 2.0 * DENS_TPB * 1.05 ? DENS_TPB2 : std::min<unsigned>(DENS_TPB, std::max(64u, half_own));
  const bool changed = b != h->block || bd != h->block_dens;
  h->block = b;
  h->block_dens = bd;
  h->blocks_from = max_own;
  return changed;
}

// k_cells: mode 0 = Verlet list build, mode 1 = the list-free per-step pass (rho, compact list, hand-out of the force pass)
// Every kernel that stages a tile in dynamic shared memory.  The opt-in to more than 48 KB belongs to the FUNCTION on the
// device, not to a handle: were it set to each handle's own size, the load of a second handle with smaller tiles would
// lower it under the first handle's launches ("invalid argument").  So every function is opened to the device's limit
// minus its own static shared memory (the mbarrier of stage_bulk, the pair-parameter table of k_force), whoever loads.
#define MDPD_UNPAREN(...) __VA_ARGS__
#define MDPD_TILE_KERNELS(X)                                                                                            \
  X((k_cells<0, false, false>), false) \
  X((k_cells<1, false, false>), false) \
  X((k_cells<1, true, false>), false) \
  X((k_cells<1, true, true>), false) \
  X((k_density<true, true, DENS_TPB>), false) \
  X((k_density<true, false, DENS_TPB>), false) \
  X((k_density<false, false, DENS_TPB>), false) \
  X((k_density<true, true, DENS_TPB2>), false) \
  X((k_density<true, false, DENS_TPB2>), false) \
  X((k_density<false, false, DENS_TPB2>), false) \
  X((k_pairs), false) \
  X((k_force<true, false>), false) \
  X((k_force<false, false>), false) \
  X((k_force<true, true>), true) \
  X((k_force<true, false, false, true>), false) \
  X((k_force<false, false, false, true>), false) \
  X((k_force<true, true, true>), true) \
  X((k_force<true, false, true>), false) \
  X((k_force<false, true>), true)

// Largest static shared memory of any tile kernel this handle can launch (the per-type-pair instantiations of the force
// pass, with their 1 KB parameter table, only when species are in use): what the capacity search has to leave free
// beside the dynamic part.
cudaError_t tile_static_smem(bool species, size_t* out) {
  size_t m = 0;
  cudaFuncAttributes a;
  cudaError_t e;
#define X(fn, multi)                                                 \
  if (species || !(multi)) {                                         \
    e = cudaFuncGetAttributes(&a, (const void*)(MDPD_UNPAREN fn));  \
    if (e != cudaSuccess) return e;                                  \
    m = std::max(m, a.sharedSizeBytes);                              \
  }
  MDPD_TILE_KERNELS(X)
#undef X
  *out = m;
  return cudaSuccess;
}

cudaError_t allow_tile_smem(mdpd_ctx* h) {
  cudaFuncAttributes a;
  cudaError_t e;
#define X(fn, multi)                                                                                                   \
  e = cudaFuncGetAttributes(&a, (const void*)(MDPD_UNPAREN fn));                                                      \
  if (e != cudaSuccess) return e;                                                                                      \
  e = cudaFuncSetAttribute((const void*)(MDPD_UNPAREN fn), cudaFuncAttributeMaxDynamicSharedMemorySize,               \
                           (int)(h->smem_limit - a.sharedSizeBytes));                                                  \
  if (e != cudaSuccess) return e;
  MDPD_TILE_KERNELS(X)
#undef X
  return cudaSuccess;
}

int launch_cells(mdpd_ctx* h, int mode, bool all, int always) {
  const DevP& d = h->d;
  const unsigned tpb = h->cells_warps[mode] * 32u;
  const size_t sm = h->smem_cells[mode];
  if (mode == 0) LAUNCH(h, PS_CELLS_LIST, (k_cells<0, false, false><<<d.ntiles, tpb, sm, h->ls>>>(d, always)));
  else if (!h->has_wall) LAUNCH(h, PS_CELLS_DIRECT, (k_cells<1, false, false><<<d.ntiles, tpb, sm, h->ls>>>(d, always)));
  else if (all) LAUNCH(h, PS_CELLS_DIRECT, (k_cells<1, true, true><<<d.ntiles, tpb, sm, h->ls>>>(d, always)));
  else LAUNCH(h, PS_CELLS_DIRECT, (k_cells<1, true, false><<<d.ntiles, tpb, sm, h->ls>>>(d, always)));
  return MDPD_OK;
}

// sort + tile recipe [+ Verlet list]: with_list = false at load time, while the tile shape is probed
int launch_rebuild_chain(mdpd_ctx* h, bool with_list = true) {
  const DevP& d = h->d;
  // grid-stride kernels on a grid of a few waves: a step whose trigger did not fire pays ~nothing for them
  const unsigned nb = std::min(nblk(h->n, TPB), 148u * 16u);
  cudaStream_t s = h->ls;
  LAUNCH(h, PS_OTHER, (k_reset_list_stats<<<1, 1, 0, s>>>(d, 0, 1)));
  LAUNCH(h, PS_CELL_COUNT, (k_cell_count<<<nb, TPB, 0, s>>>(d)));
  LAUNCH(h, PS_SCAN, (k_scan_local<<<h->L.scan_blocks, SCAN_TPB, 0, s>>>(d)));
  LAUNCH(h, PS_SCAN, (k_scan_bsum<<<1, 1024, 0, s>>>(d, h->L.scan_blocks)));
  LAUNCH(h, PS_SCAN, (k_scan_add<<<h->L.scan_blocks, SCAN_TPB, 0, s>>>(d)));
  LAUNCH(h, PS_CELL_FILL, (k_cell_fill<<<nb, TPB, 0, s>>>(d)));
  LAUNCH(h, PS_PERMUTE, (k_permute<<<nb, TPB, 0, s>>>(d)));
  LAUNCH(h, PS_RECIPE, (k_tile_recipe<<<d.ntiles, 128, 0, s>>>(d, with_list ? 1 : 0)));
  if (with_list && !h->direct) launch_cells(h, 0, false, 0);
  return MDPD_OK;
}

int launch_forces(mdpd_ctx* h, bool all, bool virial = false) {
  const DevP& d = h->d;
  if (h->direct) launch_cells(h, 1, all, 1);
  else if (h->block_dens > DENS_TPB) {
    if (!h->has_wall) LAUNCH(h, PS_DENSITY, (k_density<false, false, DENS_TPB2><<<d.ntiles, h->block_dens, h->smem_pos, h->ls>>>(d)));
    else if (all) LAUNCH(h, PS_DENSITY, (k_density<true, true, DENS_TPB2><<<d.ntiles, h->block_dens, h->smem_pos, h->ls>>>(d)));
    else LAUNCH(h, PS_DENSITY, (k_density<true, false, DENS_TPB2><<<d.ntiles, h->block_dens, h->smem_pos, h->ls>>>(d)));
  } else {
    if (!h->has_wall) LAUNCH(h, PS_DENSITY, (k_density<false, false, DENS_TPB><<<d.ntiles, h->block_dens, h->smem_pos, h->ls>>>(d)));
    else if (all) LAUNCH(h, PS_DENSITY, (k_density<true, true, DENS_TPB><<<d.ntiles, h->block_dens, h->smem_pos, h->ls>>>(d)));
    else LAUNCH(h, PS_DENSITY, (k_density<true, false, DENS_TPB><<<d.ntiles, h->block_dens, h->smem_pos, h->ls>>>(d)));
  }
  if (d.s_exp != 1.0f) {  // general exponent of wR: one material, no virial (checked by the callers)
    if (all) LAUNCH(h, PS_FORCE, (k_force<true, false, false, true><<<d.ntiles, h->block, h->smem_posvel, h->ls>>>(d)));
    else LAUNCH(h, PS_FORCE, (k_force<false, false, false, true><<<d.ntiles, h->block, h->smem_posvel, h->ls>>>(d)));
  } else if (virial) {  // mdpd_compute_virial: forces on every particle + the conservative virial tensor
    if (d.ntypes) LAUNCH(h, PS_FORCE, (k_force<true, true, true><<<d.ntiles, h->block, h->smem_posvel, h->ls>>>(d)));
    else LAUNCH(h, PS_FORCE, (k_force<true, false, true><<<d.ntiles, h->block, h->smem_posvel, h->ls>>>(d)));
  } else if (d.ntypes) {  // per-type-pair parameters
    if (all) LAUNCH(h, PS_FORCE, (k_force<true, true><<<d.ntiles, h->block, h->smem_posvel, h->ls>>>(d)));
    else LAUNCH(h, PS_FORCE, (k_force<false, true><<<d.ntiles, h->block, h->smem_posvel, h->ls>>>(d)));
  } else {
    if (all) LAUNCH(h, PS_FORCE, (k_force<true, false><<<d.ntiles, h->block, h->smem_posvel, h->ls>>>(d)));
    else LAUNCH(h, PS_FORCE, (k_force<false, false><<<d.ntiles, h->block, h->smem_posvel, h->ls>>>(d)));
  }
  return MDPD_OK;
}

int launch_integrate(mdpd_ctx* h, int do_B, int do_A, bool in_graph = false) {
  const unsigned nb = std::min(nblk(h->n, TPB), 148u * 16u);
  const int uc = in_graph ? 1 : 0;
  if (h->has_mask) LAUNCH(h, PS_INTEGRATE, (k_integrate<true><<<nb, TPB, 0, h->ls>>>(h->d, do_B, do_A, h->cond, uc)));
  else LAUNCH(h, PS_INTEGRATE, (k_integrate<false><<<nb, TPB, 0, h->ls>>>(h->d, do_B, do_A, h->cond, uc)));
  return MDPD_OK;
}

// The second half kick (Algorithm 1 line 7) of the last step is fused with the first half kick of the next one; when
// the state is read or changed between steps it is applied here.
int finalize_kick(mdpd_ctx* h) {
  if (h->pending_B && h->n) launch_integrate(h, 1, 0);
  h->pending_B = false;
  return MDPD_OK;
}

void destroy_graph(mdpd_ctx* h) {
  if (h->graph_exec) cudaGraphExecDestroy(h->graph_exec);
  if (h->graph) cudaGraphDestroy(h->graph);
  h->graph_exec = nullptr;
  h->graph = nullptr;
  h->graph_dirty = true;
}

// One timestep as a CUDA graph: k_integrate (B + A) -> IF(trigger fired){counting sort, permute, list build} ->
// k_density -> k_force.  The IF node's condition is set on the device by the last block of k_integrate, so a step whose
// trigger did not fire launches 3 kernels instead of 11 and the host never learns (or waits for) the decision.
int build_graph(mdpd_ctx* h) {
  destroy_graph(h);
  const uint64_t saved_launches = h->launches;
  cudaGraph_t g = nullptr;
  CU_TRY(h, cudaGraphCreate(&g, 0));
  h->graph = g;
  CU_TRY(h, cudaGraphConditionalHandleCreate(&h->cond, g, 0, cudaGraphCondAssignDefault));
  h->ls = h->cap_stream;
  int rc = MDPD_OK;
  do {
    if (cudaStreamBeginCaptureToGraph(h->cap_stream, g, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed) != cudaSuccess) { rc = MDPD_ECUDA; break; }
    launch_integrate(h, 1, 1, true);
    cudaStreamCaptureStatus st;
    const cudaGraphNode_t* deps = nullptr;
    size_t nd = 0;
    cudaGraph_t cg = nullptr;
    if (cudaStreamGetCaptureInfo(h->cap_stream, &st, nullptr, &cg, &deps, &nd) != cudaSuccess) { rc = MDPD_ECUDA; break; }
    cudaGraphNodeParams cp = {};
    cp.type = cudaGraphNodeTypeConditional;
    cp.conditional.handle = h->cond;
    cp.conditional.type = cudaGraphCondTypeIf;
    cp.conditional.size = 1;
    cudaGraphNode_t cn;
    if (cudaGraphAddNode(&cn, g, deps, nd, &cp) != cudaSuccess) { rc = MDPD_ECUDA; break; }
    cudaGraph_t body = cp.conditional.phGraph_out[0];
    if (cudaStreamUpdateCaptureDependencies(h->cap_stream, &cn, 1, cudaStreamSetCaptureDependencies) != cudaSuccess) { rc = MDPD_ECUDA; break; }
    launch_forces(h, false);
    cudaGraph_t out = nullptr;
    if (cudaStreamEndCapture(h->cap_stream, &out) != cudaSuccess) { rc = MDPD_ECUDA; break; }
    // the body of the IF node: the rebuild chain
    if (cudaStreamBeginCaptureToGraph(h->cap_stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed) != cudaSuccess) { rc = MDPD_ECUDA; break; }
    launch_rebuild_chain(h);
    if (cudaStreamEndCapture(h->cap_stream, &out) != cudaSuccess) { rc = MDPD_ECUDA; break; }
    if (cudaGraphInstantiate(&h->graph_exec, g, 0) != cudaSuccess) { rc = MDPD_ECUDA; break; }
  } while (0);
  h->ls = h->stream;
  h->launches = saved_launches;  // capturing launches nothing
  if (rc != MDPD_OK) {
    cudaError_t e = cudaGetLastError();
    destroy_graph(h);
    return set_err(h, rc, "building the step graph failed: %s", cudaGetErrorString(e));
  }
  h->graph_dirty = false;
  return MDPD_OK;
}

// synchronise, fetch the control block, translate latched device faults
int sync_and_check(mdpd_ctx* h) {
  CU_TRY(h, cudaMemcpyAsync(h->h_ctl, h->d.ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, h->stream));
  CU_TRY(h, cudaStreamSynchronize(h->stream));
  CU_TRY(h, cudaGetLastError());
  if (h->h_ctl->err & ERR_CHECK) return set_err(h, MDPD_ECUDA, "an internal bounds check (-DMDPD_CHECKS) failed");
  if (h->h_ctl->err & ERR_TYPE)
    return set_err(h, MDPD_EINVAL, "a particle's type is not below the number of species given to mdpd_set_pair_params");
  if (h->h_ctl->err & ERR_NAN)
    return set_err(h, MDPD_ENAN, "non-finite coordinates appeared (%llu events)", h->h_ctl->nan_events);
  if (h->h_ctl->err & ERR_TILE)
    return set_err(h, MDPD_EOVERFLOW,
                   "a tile of %d x %d x %d cells plus its halo holds %u particles, shared-memory capacity is %u "
                   "(local density too high for this tile size)",
                   h->tile_dim[0], h->tile_dim[1], h->tile_dim[2], h->h_ctl->max_halo, h->d.tile_cap);
  if (h->h_ctl->err & ERR_OVERFLOW)
    return set_err(h, MDPD_EOVERFLOW,
                   "neighbour list capacity exceeded (capacity %u, hard limit %u): raise max_neigh or lower skin",
                   h->L.cap, LCAP);
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
  h->ls = h->stream;
  if (cudaMallocHost((void**)&h->h_ctl, sizeof(Ctl)) != cudaSuccess ||
      cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
    if (h->h_ctl) cudaFreeHost(h->h_ctl);
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
  destroy_graph(h);
  if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
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
        q.max_neigh != p->max_neigh || q.mass != p->mass || q.headroom != p->headroom ||
        ((q.flags ^ p->flags) & (MDPD_FLAG_DIRECT | MDPD_FLAG_TMA_STAGING | MDPD_FLAG_CPASYNC_STAGING)))
      return set_err(h, MDPD_ESTATE, "box, cut-offs, skin, mass, capacities and the neighbour path are frozen after load_particles");
    if (p->s != 1.0f && h->ntypes) return set_err(h, MDPD_EINVAL, "per-type-pair parameters need s = 1");
    if (h->pending_B) {  // the outstanding half kick belongs to the old parameters
      CU_TRY(h, cudaSetDevice(h->device));
      finalize_kick(h);
    }
    h->prm = *p;
    fill_physics(h);
    h->graph_dirty = true;  // kernel arguments are captured by value
    return MDPD_OK;
  }
  h->prm = *p;
  h->have_params = true;
  return MDPD_OK;
}

int mdpd_set_pair_params(mdpd_ctx* h, uint32_t ntypes, const float* A, const float* B, uint32_t frozen_mask) {
  if (!h) return MDPD_EINVAL;
  if (ntypes > MAXTYPES) return set_err(h, MDPD_EINVAL, "at most %u species", MAXTYPES);
  if (ntypes && (!A || !B)) return set_err(h, MDPD_EINVAL, "A / B are NULL");
  for (uint32_t a = 0; a < ntypes; ++a)
    for (uint32_t b = 0; b < a; ++b)
      if (A[a * ntypes + b] != A[b * ntypes + a] || B[a * ntypes + b] != B[b * ntypes + a])
        return set_err(h, MDPD_EINVAL, "A and B must be symmetric");
  if (h->loaded && (ntypes != h->ntypes || frozen_mask != h->frozen_mask))
    return set_err(h, MDPD_ESTATE, "the number of species and the frozen set are fixed by load_particles");
  if (ntypes != h->ntypes) h->have_gs = false;  // the amplitude matrices belong to a species set
  h->ntypes = ntypes;
  h->frozen_mask = frozen_mask;
  for (uint32_t q = 0; q < ntypes * ntypes; ++q) {
    h->pairA[q] = A[q];
    h->pairB[q] = B[q];
  }
  if (h->loaded) {  // new values between steps: like mdpd_set_params
    CU_TRY(h, cudaSetDevice(h->device));
    if (h->pending_B) finalize_kick(h);
    fill_physics(h);
    h->graph_dirty = true;
  }
  return MDPD_OK;
}

size_t mdpd_workspace_bytes(const mdpd_params* p, uint64_t n, int has_mask, const uint32_t mask_dims[3]) {
  if (!p) return 0;
  Layout L;
  if (!make_layout(*p, n, has_mask, mask_dims, L, nullptr)) return 0;
  return L.total;
}

int mdpd_set_pair_gamma_sigma(mdpd_ctx* h, uint32_t ntypes, const float* gamma, const float* sigma) {
  if (!h) return MDPD_EINVAL;
  if (!gamma || !sigma) {
    h->have_gs = false;
  } else {
    if (ntypes == 0 || ntypes != h->ntypes)
      return set_err(h, MDPD_EINVAL, "gamma / sigma matrices need the species set of mdpd_set_pair_params (ntypes = %u there)", h->ntypes);
    for (uint32_t a = 0; a < ntypes; ++a)
      for (uint32_t b = 0; b <= a; ++b) {
        if (gamma[a * ntypes + b] != gamma[b * ntypes + a] || sigma[a * ntypes + b] != sigma[b * ntypes + a])
          return set_err(h, MDPD_EINVAL, "gamma and sigma must be symmetric");
        if (!(gamma[a * ntypes + b] >= 0.0f) || !(sigma[a * ntypes + b] >= 0.0f))
          return set_err(h, MDPD_EINVAL, "gamma and sigma must be >= 0");
      }
    for (uint32_t q = 0; q < ntypes * ntypes; ++q) {
      h->pairG[q] = gamma[q];
      h->pairS[q] = sigma[q];
    }
    h->have_gs = true;
  }
  if (h->loaded) {  // new values between steps: like mdpd_set_params
    CU_TRY(h, cudaSetDevice(h->device));
    if (h->pending_B) finalize_kick(h);
    fill_physics(h);
    h->graph_dirty = true;
  }
  return MDPD_OK;
}

int mdpd_set_workspace(mdpd_ctx* h, void* dev_ptr, size_t bytes) {
  if (!h || !dev_ptr) return MDPD_EINVAL;
  if (((uintptr_t)dev_ptr & 255u) != 0) return set_err(h, MDPD_EINVAL, "workspace must be 256-byte aligned");
  if (h->loaded) {  // a new workspace drops the loaded state: the next call must be mdpd_load_particles
    cudaSetDevice(h->device);
    cudaStreamSynchronize(h->stream);
    destroy_graph(h);
    h->loaded = false;
    h->pending_B = false;
  }
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
  if (h->prm.s != 1.0f && h->ntypes) return set_err(h, MDPD_EINVAL, "per-type-pair parameters need s = 1");
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
  if (h->ws_owned && h->ws_bytes < L.total) {  // the library's own allocation grows with the problem
    CU_TRY(h, cudaStreamSynchronize(h->stream));
    destroy_graph(h);
    cudaFree(h->ws);
    h->ws = nullptr;
    h->ws_bytes = L.total + (64u << 20);
    CU_TRY(h, cudaMalloc((void**)&h->ws, h->ws_bytes));
  }
  if (h->ws_bytes < L.total)
    return set_err(h, MDPD_ENOMEM, "workspace too small: %zu bytes given, %zu needed", h->ws_bytes, L.total);
  h->mask_cap = h->ws_bytes - L.mask;
  h->L = L;
  h->n = n;
  h->has_mask = false;
  h->loaded = false;
  h->pending_B = false;
  h->graph_dirty = true;
  fill_devp(h);
  fill_physics(h);
  h->host_step = 0;
  {
    int v = 0;
    CU_TRY(h, cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, h->device));
    h->smem_limit = (size_t)v;
  }
  CU_TRY(h, cudaMemsetAsync(h->d.ctl, 0, sizeof(Ctl), h->stream));
  if (n) {
    char* st = h->ws + L.stage;
    float* spos = (float*)st;
    float* svel = spos + 3 * n;
    unsigned char* stype = (unsigned char*)(svel + 3 * n);
    CU_TRY(h, cudaMemcpyAsync(spos, pos, n * 12, cudaMemcpyDefault, h->stream));
    CU_TRY(h, cudaMemcpyAsync(svel, vel, n * 12, cudaMemcpyDefault, h->stream));
    if (type) CU_TRY(h, cudaMemcpyAsync(stype, type, n, cudaMemcpyDefault, h->stream));
    LAUNCH(h, PS_OTHER, (k_pack<<<nblk(n, TPB), TPB, 0, h->stream>>>(h->d, spos, svel, type ? stype : nullptr, 0u)));
  }
  {
    int v = 0;
    CU_TRY(h, cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, h->device));
    h->d.sms = (unsigned)v;
  }
  h->direct = (h->prm.flags & MDPD_FLAG_DIRECT) != 0;
  // chosen by measurement (profiles/r2_staging.md): bulk copies win in the density pass, per-particle cp.async in the force pass
  h->d.tma_staging = (h->prm.flags & MDPD_FLAG_TMA_STAGING) ? 3u : ((h->prm.flags & MDPD_FLAG_CPASYNC_STAGING) ? 0u : 1u);
  h->chain_launches = h->direct ? 8u : 9u;  // reset, count, 3 x scan, fill, permute, recipe [, list]
  // Tile shape: the largest candidate that still gives every SM work and whose most populated tile + halo fits in
  // shared memory (checked on the device after the sort).
  static const int kCand[][3] = {{4, 4, 4}, {4, 4, 2}, {4, 2, 2}, {2, 2, 2}, {2, 2, 1}, {2, 1, 1}, {1, 1, 1}};
  const int ncand = (int)(sizeof kCand / sizeof kCand[0]);
#ifndef MDPD_FIRST_TILE
#define MDPD_FIRST_TILE 0  // measurement builds: start the search at a smaller tile shape (profiles/r2_experiments.md)
#endif
  int first = MDPD_FIRST_TILE;
  {
    auto ntiles_of = [&](const int* t) {
      return (size_t)((L.ncx + t[0] - 1) / t[0]) * ((L.ncy + t[1] - 1) / t[1]) * ((L.ncz + t[2] - 1) / t[2]);
    };
    while (first < 3 && ntiles_of(kCand[first]) < 148) ++first;  // small boxes: down to 2 x 2 x 2
  }
  for (int ci = first; ci < ncand; ++ci) {
    const int* cand = kCand[ci];
    int tdim[3] = {std::min<int>(cand[0], (int)L.ncx), std::min<int>(cand[1], (int)L.ncy), std::min<int>(cand[2], (int)L.ncz)};
    std::vector<unsigned> rank;
    std::vector<TileInfo> tiles;
    build_tile_ranks(L, tdim, rank, tiles);
    memcpy(h->tile_dim, tdim, sizeof tdim);
    h->d.ntiles = (unsigned)tiles.size();
    h->d.nrun_max = 3u * (unsigned)((tdim[1] + 2) * (tdim[2] + 2));
    h->d.hb_off = 1u + h->d.nrun_max;
    h->d.run_stride = h->d.hb_off + ((unsigned)((tdim[0] + 2) * (tdim[1] + 2) * (tdim[2] + 2)) + 1u + 7u) / 8u;
    if ((size_t)h->d.ntiles * h->d.run_stride > (size_t)L.ncell * 32 + 4096)
      return set_err(h, MDPD_ENOMEM, "tile recipe table does not fit its reservation");
    h->block = TILE_TPB;  // upper bound while the capacity is probed; set from the tile population below
    {  // slack of k_cells' approximate range test: its rounding error grows with the square of the centred coordinates
      double x2 = 0.0;
      for (int k = 0; k < 3; ++k) {
        const double edge = (double)h->prm.box[k] / (double)(k == 0 ? L.ncx : (k == 1 ? L.ncy : L.ncz));
        const double x = 0.5 * tdim[k] * edge + edge + 0.5 * (double)h->prm.skin + 1.0 / 32.0;
        x2 += x * x;
      }
      h->d.dot_margin = (float)(6e-6 * x2);
    }
    // fixed part of a tile kernel's shared memory: tables of the staged image + the largest static allocation of any of them
    size_t stat = 0;
    CU_TRY(h, tile_static_smem(h->ntypes != 0, &stat));
    const size_t fixed = tile_smem_bytes(0, true, 0) + stat;
    // capacity of a tile + halo in staged slots: what the force pass can hold in shared memory, what a 16-bit list entry can
    // address, and what the item list of stage_fast (2 * HTAB items: 3 * 36 runs + one item per 32 slots) can describe
    const unsigned cap_limit = (unsigned)std::min<size_t>(std::min<size_t>((h->smem_limit - fixed) / TILE_SLOT_BYTES, 65535),
                                                          (size_t)(2 * HTAB - 3 * 36) * 32);
    h->d.tile_cap = cap_limit;
    LAUNCH(h, PS_OTHER, (k_ctl_init<<<1, 1, 0, h->stream>>>(h->d)));  // the initial sort reads buffer 0 and writes buffer 1
    CU_TRY(h, cudaMemcpyAsync(h->d.cell_rank, rank.data(), rank.size() * 4, cudaMemcpyHostToDevice, h->stream));
    CU_TRY(h, cudaMemcpyAsync((void*)h->d.tiles, tiles.data(), tiles.size() * sizeof(TileInfo), cudaMemcpyHostToDevice,
                              h->stream));
    CU_TRY(h, cudaMemsetAsync(h->d.cell_count, 0, (size_t)L.ncell * 4, h->stream));
    if (n) launch_rebuild_chain(h, false);  // sort + tile statistics, no list yet
    CU_TRY(h, cudaMemcpyAsync(h->h_ctl, h->d.ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, h->stream));
    CU_TRY(h, cudaStreamSynchronize(h->stream));  // rank, tiles are locals
    h->has_wall = h->h_ctl->has_wall != 0;
    const unsigned max_halo = h->h_ctl->max_halo;
    const double headroom = h->prm.headroom > 0.0f ? std::max(1.0, (double)h->prm.headroom) : 1.15;  // mdpd_params.headroom
    if ((double)max_halo * headroom > (double)cap_limit) {
      if (ci + 1 == ncand)
        return set_err(h, MDPD_EOVERFLOW, "a tile of %d x %d x %d cells plus halo holds %u particles (x head-room %.2f); shared memory fits %u",
                       tdim[0], tdim[1], tdim[2], max_halo, headroom, cap_limit);
      continue;  // try the next smaller tile shape
    }
    choose_blocks(h, h->h_ctl->max_own);
    // head-room for density fluctuations between rebuilds of a long run
    {
      // at least `headroom` (default 15 %) over the fullest tile of the initial state; beyond that, all the shared memory that does not
      // cost a resident CTA of the force pass (the tightest: it stages positions and velocities)
      unsigned want = std::min<unsigned>(cap_limit, ((unsigned)(max_halo * headroom) + 64 + 63) / 64 * 64);
      const size_t sm_total = h->smem_limit + 1024;  // per-SM shared memory; 1 KB is reserved per resident CTA
      if (!(h->prm.headroom > 0.0f)) {
        // default head-room: 15 %, but no less than 8 % where the difference decides whether two CTAs of the force pass fit per SM
        // (3.4 against 2.5 ms per launch on config 4a just above the limit; profiles/r2_experiments.md section 5)
        const size_t half = sm_total / 2;
        const unsigned two = half > 1024 + fixed ? (unsigned)((half - 1024 - fixed) / TILE_SLOT_BYTES / 64 * 64) : 0u;
        if (want > two && (double)max_halo * 1.08 + 64.0 <= (double)two) want = two;
      }
      const size_t per_cta = tile_smem_bytes(want, true, 0) + stat + 1024;
      const size_t ctas = std::max<size_t>(1, sm_total / per_cta);
      const size_t room = sm_total / ctas - 1024 - fixed;
      // ... nor one of the density pass (positions only, DENS_MINB CTAs per SM) or of the list build (two): when the force pass is
      // down to one CTA per SM the capacity must not grow into the other passes' occupancy
      const auto slots_for = [&](size_t n_ctas, size_t slot_bytes, size_t extra) {
        const size_t per = sm_total / n_ctas;
        const size_t fix = 1024 + tile_smem_bytes(0, false, 0) + stat + extra;
        return per > fix ? (per - fix) / slot_bytes : 0;
      };
      const size_t grow = std::min(std::min<size_t>(room / TILE_SLOT_BYTES, slots_for(DENS_MINB, 16, 0)),
                                   slots_for(2, 16, HTAB * 2 + (size_t)CELLS_MAXW0 * CELLS_ROW0_BYTES));
      h->d.tile_cap = std::max<unsigned>(want, std::min<unsigned>(cap_limit, (unsigned)(grow / 64 * 64)));
    }
    break;
  }
  h->smem_pos = tile_smem_bytes(h->d.tile_cap, false, 0);
  h->smem_posvel = tile_smem_bytes(h->d.tile_cap, true, 0);
  // k_cells: the staged image plus one row buffer (32 rows) per warp; as many warps as two resident CTAs per SM allow
  h->d.cap_act = L.cap_act;
  h->d.rows_verlet = cells_row_bytes(h->d.cap);
  h->d.rows_direct = cells_row_bytes(h->d.cap_act);
  for (int mode = 0; mode < 2; ++mode) {
    const size_t rowb = mode ? 32 * (size_t)h->d.rows_direct + 64 : (size_t)CELLS_ROW0_BYTES;
    const size_t base = cells_smem_bytes(h->d.tile_cap, 0, 0);
    const size_t two = (h->smem_limit + 1024) / 2 - 1024;  // per CTA when two are resident
    size_t nw = two > base ? (two - base) / rowb : 0;
    if (nw < 4) nw = h->smem_limit > base ? (h->smem_limit - base) / rowb : 0;  // one resident CTA
    if (nw < 1) return set_err(h, MDPD_ENOMEM, "k_cells: the staged tile and one row buffer do not fit in shared memory");
    h->cells_warps[mode] = (unsigned)std::min<size_t>(nw, mode ? CELLS_MAXW : CELLS_MAXW0);
    h->smem_cells[mode] = base + h->cells_warps[mode] * rowb;
  }
  CU_TRY(h, allow_tile_smem(h));
  if (n) {
    // the recipe again, now against the final capacity (a tile that does not fit is flagged), then the list and the forces
    LAUNCH(h, PS_RECIPE, (k_tile_recipe<<<h->d.ntiles, 128, 0, h->stream>>>(h->d, 1)));
    if (!h->direct) launch_cells(h, 0, false, 1);
    launch_forces(h, true);
  }
  h->loaded = true;
  return sync_and_check(h);
}

int mdpd_load_wall_mask(mdpd_ctx* h, const uint8_t* mask, const uint32_t dims[3], float voxel) {
  if (!h) return MDPD_EINVAL;
  if (!h->loaded) return set_err(h, MDPD_ESTATE, "load_particles first");
  CU_TRY(h, cudaSetDevice(h->device));
  h->graph_dirty = true;
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
  if (h->h_ctl->max_own && h->h_ctl->max_own != h->blocks_from && choose_blocks(h, h->h_ctl->max_own)) h->graph_dirty = true;
  const bool graphs = h->use_graph && !h->prof_on && !(h->prm.flags & MDPD_FLAG_NO_GRAPH);
  if (graphs && h->graph_dirty && (nsteps > 1 || h->pending_B)) {
    int rc = build_graph(h);
    if (rc != MDPD_OK) return rc;
  }
  for (uint32_t it = 0; it < nsteps; ++it) {
    if (graphs && h->pending_B) {  // steady state: one graph replay per step
      CU_TRY(h, cudaGraphLaunch(h->graph_exec, h->stream));
      h->graph_steps += 1;
    } else {
      // [second half kick of the previous step +] half kick, drift, bounce, trigger
      launch_integrate(h, h->pending_B ? 1 : 0, 1);
      launch_rebuild_chain(h);   // every kernel returns at once unless the trigger fired (device-side predicate)
      launch_forces(h, false);   // Algorithm 1 lines 4 and 6 at the new time level, half-step velocities
    }
    h->pending_B = true;         // Algorithm 1 line 7 is fused into the next step (or applied by finalize_kick)
  }
  CU_TRY(h, cudaGetLastError());
  return MDPD_OK;
}

int mdpd_compute_forces(mdpd_ctx* h) {
  if (!h) return MDPD_EINVAL;
  if (!h->loaded) return set_err(h, MDPD_ESTATE, "load_particles first");
  if (h->n == 0) return MDPD_OK;
  CU_TRY(h, cudaSetDevice(h->device));
  finalize_kick(h);
  launch_forces(h, true);
  return sync_and_check(h);
}

int mdpd_compute_virial(mdpd_ctx* h, double out[6]) {
  if (!h || !out) return MDPD_EINVAL;
  if (!h->loaded) return set_err(h, MDPD_ESTATE, "load_particles first");
  for (int k = 0; k < 6; ++k) out[k] = 0.0;
  if (h->n == 0) return MDPD_OK;
  CU_TRY(h, cudaSetDevice(h->device));
  finalize_kick(h);
  if (h->prm.s != 1.0f) return set_err(h, MDPD_EINVAL, "mdpd_compute_virial needs s = 1");
  CU_TRY(h, cudaMemsetAsync(h->d.ctl->vir, 0, sizeof(double) * 6, h->stream));
  launch_forces(h, true, true);
  int rc = sync_and_check(h);
  for (int k = 0; k < 6; ++k) out[k] = 0.5 * h->h_ctl->vir[k];  // the full list visits every pair from both ends
  return rc;
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

int mdpd_set_forces(mdpd_ctx* h, const float* force) {
  if (!h) return MDPD_EINVAL;
  if (!h->loaded) return set_err(h, MDPD_ESTATE, "load_particles first");
  if (h->n == 0) return MDPD_OK;
  if (!force) return set_err(h, MDPD_EINVAL, "force is NULL");
  CU_TRY(h, cudaSetDevice(h->device));
  finalize_kick(h);
  float* sf = (float*)(h->ws + h->L.stage);
  CU_TRY(h, cudaMemcpyAsync(sf, force, h->n * 12, cudaMemcpyDefault, h->stream));
  LAUNCH(h, PS_OTHER, (k_set_forces<<<nblk(h->n, TPB), TPB, 0, h->stream>>>(h->d, sf)));
  return sync_and_check(h);
}

int mdpd_get_state(mdpd_ctx* h, float* pos, float* vel, float* force, float* rho, uint64_t* step) {
  if (!h) return MDPD_EINVAL;
  if (!h->loaded) return set_err(h, MDPD_ESTATE, "load_particles first");
  CU_TRY(h, cudaSetDevice(h->device));
  const uint64_t n = h->n;
  finalize_kick(h);
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

int mdpd_get_counters(mdpd_ctx* h, uint64_t out[MDPD_NCOUNTERS]) {
  if (!h || !out) return MDPD_EINVAL;
  if (!h->loaded) return set_err(h, MDPD_ESTATE, "load_particles first");
  CU_TRY(h, cudaSetDevice(h->device));
  int rc = sync_and_check(h);
  const Ctl* c = h->h_ctl;
  for (int k = 0; k < MDPD_NCOUNTERS; ++k) out[k] = 0;
  out[0] = h->host_step;
  out[1] = c->rebuilds;
  out[2] = c->bounces;
  out[3] = c->max_nbr;
  out[4] = c->sum_nbr;
  out[5] = c->max_halo;
  out[6] = c->overflow + c->nan_events;
  out[7] = h->launches + 3 * h->graph_steps + h->chain_launches * c->graph_rebuilds;  // a graph replay launches 3 kernels (+ the rebuild chain)
  out[8] = c->sum_act;
  out[9] = c->dens_passes;
  out[10] = (uint64_t)h->tile_dim[0] | ((uint64_t)h->tile_dim[1] << 8) | ((uint64_t)h->tile_dim[2] << 16);
  out[11] = h->d.ntiles;
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
  if (h->direct) {  // the list-free path keeps no Verlet list: build one from the current cells for this call
    LAUNCH(h, PS_OTHER, (k_reset_list_stats<<<1, 1, 0, h->stream>>>(h->d, 1, 0)));
    launch_cells(h, 0, false, 1);
  }
  LAUNCH(h, PS_OTHER, (k_pairs<<<h->d.ntiles, h->block, h->smem_pos, h->stream>>>(h->d, rcut * rcut, dout, cap, dcnt)));
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

// mdpd_get_pairs for callers that cannot allocate device memory (see include/mdpd.h): same kernel, same result,
// but the counter and the pair buffer live in g_pairs_scratch instead of two cudaMalloc blocks.  Nothing in here calls
// cudaMalloc / cudaFree or a routine that allocates behind the caller's back: the copies go through the runtime's
// own staging, the sort is in place.
int mdpd_get_pairs_static(mdpd_ctx* h, float rcut, uint64_t* count, uint32_t* pairs, uint64_t cap) {
  if (!h || !count) return MDPD_EINVAL;
  if (!h->loaded) return set_err(h, MDPD_ESTATE, "load_particles first");
  if (!(rcut > 0) || rcut > h->L.rlist) return set_err(h, MDPD_EINVAL, "rcut must be in (0, rc + skin]");
  if (!pairs) cap = 0;
  if (cap > (uint64_t)MDPD_STATIC_PAIRS_MAX)
    return set_err(h, MDPD_EINVAL,
                   "mdpd_get_pairs_static: cap = %llu pairs does not fit the fixed scratch array (MDPD_STATIC_PAIRS_MAX = %u "
                   "pairs); ask for fewer pairs or use mdpd_get_pairs, which allocates",
                   (unsigned long long)cap, (unsigned)MDPD_STATIC_PAIRS_MAX);
  if (h->prof_on)  // the per-kernel timing creates CUDA events on demand, which this entry point promises not to do
    return set_err(h, MDPD_ESTATE, "mdpd_get_pairs_static: not between mdpd_profile_begin and mdpd_profile_end");
  CU_TRY(h, cudaSetDevice(h->device));
  *count = 0;
  if (h->n == 0) return MDPD_OK;
  unsigned char* base = nullptr;
  {
    cudaError_t e = static_pairs_scratch(h->device, &base);  // first call on this device: resolves the address
    if (e != cudaSuccess)
      return set_err(h, MDPD_ECUDA, "mdpd_get_pairs_static: cudaGetSymbolAddress of the scratch array failed: %s",
                     cudaGetErrorString(e));
  }
  unsigned long long* dcnt = (unsigned long long*)base;
  uint2* dout = (uint2*)(base + STATIC_PAIRS_HEAD);
  // The array still holds whatever the previous call left.  Only the counter has to start at zero: the pair slots
  // below the new count are all rewritten, the ones above it are never read.
  CU_TRY(h, cudaMemsetAsync(dcnt, 0, sizeof(unsigned long long), h->stream));
  if (h->direct) {  // the list-free path keeps no Verlet list: build one from the current cells (workspace memory only)
    LAUNCH(h, PS_OTHER, (k_reset_list_stats<<<1, 1, 0, h->stream>>>(h->d, 1, 0)));
    launch_cells(h, 0, false, 1);
  }
  LAUNCH(h, PS_OTHER, (k_pairs<<<h->d.ntiles, h->block, h->smem_pos, h->stream>>>(h->d, rcut * rcut, dout, cap, dcnt)));
  CU_TRY(h, cudaGetLastError());
  unsigned long long c = 0;
  CU_TRY(h, cudaMemcpyAsync(&c, dcnt, sizeof c, cudaMemcpyDeviceToHost, h->stream));
  CU_TRY(h, cudaStreamSynchronize(h->stream));
  if (cap) {
    const uint64_t m = std::min<uint64_t>(c, cap);
    CU_TRY(h, cudaMemcpyAsync(pairs, dout, m * sizeof(uint2), cudaMemcpyDeviceToHost, h->stream));
    CU_TRY(h, cudaStreamSynchronize(h->stream));
    struct TagPair { uint32_t a, b; };  // same bytes as the caller's [m][2] uint32 rows
    TagPair* tp = reinterpret_cast<TagPair*>(pairs);
    std::sort(tp, tp + m, [](const TagPair& x, const TagPair& y) { return x.a != y.a ? x.a < y.a : x.b < y.b; });
  }
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

#ifndef MDPD_BUILD_FLAGS
#define MDPD_BUILD_FLAGS ""
#endif
const char* mdpd_build_flags(void) { return MDPD_BUILD_FLAGS; }

const char* mdpd_profile_name(int slot) { return (slot >= 0 && slot < PS_COUNT) ? kProfNames[slot] : ""; }

int mdpd_probe_issue_rates(int device, void* cuda_stream, double out[4]) {
  if (!out) return MDPD_EINVAL;
  for (int k = 0; k < 4; ++k) out[k] = 0.0;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int sms = 0, khz = 0;
  if (cudaSetDevice(device) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess ||
      cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, device) != cudaSuccess)
    return MDPD_ECUDA;
  float* sink = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (cudaMalloc((void**)&sink, 4) != cudaSuccess) return MDPD_ECUDA;
  int rc = MDPD_OK;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) rc = MDPD_ECUDA;
  const int blocks = sms * 2;  // 2 x 1024 threads = 64 resident warps per SM
  const double per_iter[3] = {1.0, 2.0, 2.0};  // warp instructions per chain and iteration (FFMA; LOP3 + VIMNMX; IMAD.WIDE + IADD)
  for (int kind = 0; kind < 3 && rc == MDPD_OK; ++kind) {
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {  // the first repetition warms up
      cudaEventRecord(e0, st);
      if (kind == 0) k_probe<0><<<blocks, PROBE_TPB, 0, st>>>(sink, 1.0001f, 0.5f, 0x9E3779B9u, 0x12345u);
      if (kind == 1) k_probe<1><<<blocks, PROBE_TPB, 0, st>>>(sink, 1.0001f, 0.5f, 0x9E3779B9u, 0x12345u);
      if (kind == 2) k_probe<2><<<blocks, PROBE_TPB, 0, st>>>(sink, 1.0001f, 0.5f, 0x9E3779B9u, 0x12345u);
      cudaEventRecord(e1, st);
      if (cudaEventSynchronize(e1) != cudaSuccess) { rc = MDPD_ECUDA; break; }
      float ms = 0.f;
      cudaEventElapsedTime(&ms, e0, e1);
      if (rep > 0 && ms < best) best = ms;
    }
    const double winst = (double)blocks * (PROBE_TPB / 32) * PROBE_ITER * PROBE_CH * per_iter[kind];
    out[kind] = winst / ((double)best * 1e-3);
  }
  out[3] = (double)khz * 1e3;
  if (cudaGetLastError() != cudaSuccess) rc = MDPD_ECUDA;
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  cudaFree(sink);
  return rc;
}

}  // extern "C"
