// tfa_solve.cu — the linear solve of Eq. 14 (L123) on the assembled BSR system: BSR
// matrix-vector product, block-Jacobi preconditioner, restarted GMRES (the paper's solver configuration,
// L28, L392).  Kernels are HBM-bound streams; the Hessenberg least-squares problem lives on the host.
#include <algorithm>
#include <cmath>
#include <functional>
#include <vector>

#include "tfa_common.cuh"
#include "tfa_tma.cuh"

namespace tfa {
int assemble_impl(tfa_ctx* ctx, const tfa_mesh* m, const double* state, const double* state_n,
                  const double* state_nm1, double dt, double* rhs, double* bsr_vals, void* stream, bool timed,
                  int phases = 3, double* offd_vals = nullptr);

constexpr int SV_CELLS = 16;              // cells per CTA: thread = (cell, scalar row)
constexpr int SV_T = SV_CELLS * NEQ;      // 288 threads
constexpr int MAXK = 64;                  // largest restart length

// ------------------------------------------------------------------------------------------------
// y = A x: thread (i, r) walks the blocks of BSR row i and reads scalar row r of each block (18 contiguous
// doubles; the 18 threads of a cell read the whole 2592-byte block contiguously).  Algorithmic bytes =
// the matrix (2592 per block) + x + y: HBM-bound.  With DIAG_ONLY the "matrix" is the block-diagonal
// dinv [nc][18][18] (the preconditioner's application).
// ------------------------------------------------------------------------------------------------
template <bool DIAG_ONLY>
__global__ void __launch_bounds__(SV_T) k_bsr_spmv(int64_t nc, const int32_t* __restrict__ rowptr,
                                                  const int32_t* __restrict__ col, const double* __restrict__ vals,
                                                  const double* __restrict__ x, double* __restrict__ y) {
  const int r = threadIdx.x % NEQ;
  const int64_t i = blockIdx.x * (int64_t)SV_CELLS + threadIdx.x / NEQ;
  if (i >= nc) return;
  const int64_t b0 = DIAG_ONLY ? i : rowptr[i], b1 = DIAG_ONLY ? i + 1 : rowptr[i + 1];
  double acc = 0.0;
  for (int64_t b = b0; b < b1; ++b) {
    const int64_t j = DIAG_ONLY ? i : col[b];
    const double2* __restrict__ a = reinterpret_cast<const double2*>(vals + b * BLK + r * NEQ);
    const double2* __restrict__ xv = reinterpret_cast<const double2*>(x + NEQ * j);
#pragma unroll
    for (int c = 0; c < NEQ / 2; ++c) {
      const double2 av = a[c], xx = xv[c];
      acc = fma(av.x, xx.x, acc);
      acc = fma(av.y, xx.y, acc);
    }
  }
  y[NEQ * i + r] = acc;
}

// ------------------------------------------------------------------------------------------------
// The same product on the packed Jacobian (tfa.h TFA_PACKED_BLOCK): thread (i, r) reads row r of the diagonal block
// and, of every off-diagonal block of the row, the 8 (field rows) or 5 (species rows) entries of its group's
// sub-block; 5328 instead of 10368 matrix bytes per triangle.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void packed_row(int r, int& base, int& n, int& c0, int& cs, int& cT) {
  // row r of the 18-vector -> start of its sub-block row inside a packed block, the number of columns n, and the
  // columns: fields 0..7; species s: rho 8+s, u 10+3s .. 12+3s, T 16+s
  if (r < 8) { base = 8 * r; n = 8; c0 = 0; cs = 0; cT = 0; return; }
  const int s = r == 9 || (r >= 13 && r <= 15) || r == 17;
  const int q = (r == 8 + s) ? 0 : (r == 16 + s ? 4 : r - (9 + 3 * s));
  base = 64 + 25 * s + 5 * q;
  n = 5;
  c0 = 8 + s;
  cs = 10 + 3 * s;
  cT = 16 + s;
}
// The off-diagonal blocks of a CTA's 16 rows are one contiguous piece of the packed array (BSR order with the
// diagonal blocks taken out): it comes in by TMA, one bulk copy per row, while the threads do the diagonal blocks,
// and is read from shared memory -- 16-byte loads for the field rows, whose 8 entries start on a 64-byte boundary.
// (Before: 8-byte global loads, 64 or 40 bytes apart between the threads of a cell: four times the sectors in L1
// requests, 1.18 ms = 0.74 of HBM at c4b.)
__global__ void __launch_bounds__(SV_T) k_packed_spmv(int64_t nc, int BS, const int32_t* __restrict__ rowptr,
                                                     const int32_t* __restrict__ col, const int32_t* __restrict__ blkmap,
                                                     const double* __restrict__ dvals, const double* __restrict__ ovals,
                                                     const double* __restrict__ x, double* __restrict__ y) {
  extern __shared__ __align__(128) unsigned char ps_raw[];
  double* const sm = reinterpret_cast<double*>(ps_raw + 16);
  uint64_t* const bar = reinterpret_cast<uint64_t*>(ps_raw);
  const int r = threadIdx.x % NEQ;
  const int64_t i0 = blockIdx.x * (int64_t)SV_CELLS, i = i0 + threadIdx.x / NEQ;
  const int64_t iend = min(i0 + SV_CELLS, nc);
  const int64_t s0 = rowptr[i0] - i0;   // the CTA's first off-diagonal slot
  if (threadIdx.x == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    mbar_arrive_expect_tx(bar, (uint32_t)((rowptr[iend] - iend - s0) * (TFA_PACKED_BLOCK * sizeof(double))));
  }
  __syncthreads();
  const bool live = i < nc;
  int64_t b0 = 0, b1 = 0;
  if (live) {
    b0 = rowptr[i];
    b1 = rowptr[i + 1];
    if (r == 0 && b1 - b0 > 1)
      bulk_load(sm + (b0 - i - s0) * TFA_PACKED_BLOCK, ovals + (b0 - i) * TFA_PACKED_BLOCK,
                (uint32_t)((b1 - b0 - 1) * (TFA_PACKED_BLOCK * sizeof(double))), bar);
  }
  double acc = 0.0;
  if (live) {
    const double2* __restrict__ a = reinterpret_cast<const double2*>(dvals + i * BLK + r * NEQ);
    const double2* __restrict__ xv = reinterpret_cast<const double2*>(x + NEQ * i);
#pragma unroll
    for (int c = 0; c < NEQ / 2; ++c) {
      const double2 av = a[c], xx = xv[c];
      acc = fma(av.x, xx.x, acc);
      acc = fma(av.y, xx.y, acc);
    }
  }
  mbar_wait(bar, 0);
  if (!live) return;
  int base, n, c0, cs, cT;
  packed_row(r, base, n, c0, cs, cT);
  const int64_t bd = blkmap[(int64_t)BS * i];
  const double* __restrict__ a = sm + (b0 - i - s0) * TFA_PACKED_BLOCK + base;
  for (int64_t b = b0; b < b1; ++b) {
    if (b == bd) continue;
    const double* __restrict__ xj = x + NEQ * (int64_t)col[b];
    if (n == 8) {
      const double2* __restrict__ a2 = reinterpret_cast<const double2*>(a);
      const double2* __restrict__ x2 = reinterpret_cast<const double2*>(xj);
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        const double2 av = a2[c], xx = x2[c];
        acc = fma(av.y, xx.y, fma(av.x, xx.x, acc));
      }
    } else {
      acc = fma(a[0], xj[c0], acc);
      acc = fma(a[1], xj[cs], acc);
      acc = fma(a[2], xj[cs + 1], acc);
      acc = fma(a[3], xj[cs + 2], acc);
      acc = fma(a[4], xj[cT], acc);
    }
    a += TFA_PACKED_BLOCK;
  }
  y[NEQ * i + r] = acc;
}
// dynamic shared memory of k_packed_spmv: the off-diagonal blocks of SV_CELLS rows of F faces, and the mbarrier
static size_t packed_spmv_smem(int F) { return 16 + sizeof(double) * SV_CELLS * F * TFA_PACKED_BLOCK; }
static int launch_packed_spmv(const tfa_mesh* m, const double* dvals, const double* ovals, const double* x, double* y,
                              cudaStream_t st) {
  if ((reinterpret_cast<uintptr_t>(dvals) | reinterpret_cast<uintptr_t>(ovals) | reinterpret_cast<uintptr_t>(x)) & 15)
    return set_error(TFA_EINVAL, "tfa_packed_spmv: the packed arrays and x must be 16-byte aligned");
  TFA_CUDA(cudaFuncSetAttribute(k_packed_spmv, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)packed_spmv_smem(4)));
  k_packed_spmv<<<cdiv(m->nc, SV_CELLS), SV_T, packed_spmv_smem(m->F), st>>>(
      m->nc, blk_stride(m->F), m->bsr_rowptr.p, m->bsr_col.p, m->blkmap.p, dvals, ovals, x, y);
  return 0;
}

// ------------------------------------------------------------------------------------------------
// Mixed precision (tfa_gmres_packed_f32): the packed Jacobian and the block-diagonal preconditioner stored in FP32,
// vectors and accumulation in FP64.  Off-diagonal blocks sit TFA_PACKED_BLOCK_F32 = 116 floats apart (464 bytes: a
// 16-byte multiple, so that a row's blocks can come in by TMA and the field rows be read with 16-byte loads).
// ------------------------------------------------------------------------------------------------
constexpr int PKF = TFA_PACKED_BLOCK_F32;
__global__ void k_to_f32(int64_t n, const double* __restrict__ src, float* __restrict__ dst) {
  for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < n; e += (int64_t)blockDim.x * gridDim.x)
    dst[e] = (float)src[e];
}
__global__ void k_offd_to_f32(int64_t nblk, const double* __restrict__ src, float* __restrict__ dst) {
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < nblk * PKF; t += (int64_t)blockDim.x * gridDim.x) {
    const int64_t b = t / PKF;
    const int e = (int)(t - b * PKF);
    dst[t] = e < TFA_PACKED_BLOCK ? (float)src[b * TFA_PACKED_BLOCK + e] : 0.0f;
  }
}
__global__ void __launch_bounds__(SV_T) k_packed_spmv_f32(int64_t nc, int BS, int maxrow,
                                                         const int32_t* __restrict__ rowptr,
                                                         const int32_t* __restrict__ col,
                                                         const int32_t* __restrict__ blkmap,
                                                         const float* __restrict__ dvals, const float* __restrict__ ovals,
                                                         const double* __restrict__ x, double* __restrict__ y) {
  // shared memory: mbarrier | x rows of every block of the CTA's rows (diagonal ones included), 18 doubles each |
  // the off-diagonal blocks (FP32, PKF apart)
  extern __shared__ __align__(128) unsigned char ps_raw[];
  uint64_t* const bar = reinterpret_cast<uint64_t*>(ps_raw);
  double* const xs = reinterpret_cast<double*>(ps_raw + 16);
  const int maxblk = SV_CELLS * maxrow;   // maxrow = F + 1 blocks per row at most
  float* const sm = reinterpret_cast<float*>(ps_raw + 16 + sizeof(double) * NEQ * maxblk);
  const int r = threadIdx.x % NEQ;
  const int64_t i0 = blockIdx.x * (int64_t)SV_CELLS, i = i0 + threadIdx.x / NEQ;
  const int64_t iend = min(i0 + SV_CELLS, nc);
  const int64_t B0 = rowptr[i0], B1 = rowptr[iend];
  const int64_t s0 = B0 - i0;   // the CTA's first off-diagonal slot
  if (threadIdx.x == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    mbar_arrive_expect_tx(bar, (uint32_t)((B1 - iend - s0) * (PKF * sizeof(float))));
  }
  __syncthreads();
  const bool live = i < nc;
  int64_t b0 = 0, b1 = 0;
  if (live) {
    b0 = rowptr[i];
    b1 = rowptr[i + 1];
    if (r == 0 && b1 - b0 > 1)
      bulk_load(sm + (b0 - i - s0) * PKF, ovals + (b0 - i) * PKF, (uint32_t)((b1 - b0 - 1) * (PKF * sizeof(float))), bar);
  }
  // the x rows the CTA multiplies with, gathered once (16-byte pieces, nine per row) instead of once per thread
  {
    const int npieces = (int)(B1 - B0) * (NEQ / 2);
    double2* __restrict__ xs2 = reinterpret_cast<double2*>(xs);
    const double2* __restrict__ x2 = reinterpret_cast<const double2*>(x);
    for (int q = threadIdx.x; q < npieces; q += SV_T) {
      const int blk = q / (NEQ / 2), piece = q - blk * (NEQ / 2);
      xs2[q] = x2[(int64_t)col[B0 + blk] * (NEQ / 2) + piece];
    }
  }
  double acc = 0.0;
  int base, n, c0, cs, cT;
  packed_row(r, base, n, c0, cs, cT);
  __syncthreads();
  if (live) {
    const int64_t bd = blkmap[(int64_t)BS * i];
    const float2* __restrict__ a = reinterpret_cast<const float2*>(dvals + i * BLK + r * NEQ);
    const double2* __restrict__ xv = reinterpret_cast<const double2*>(xs + NEQ * (bd - B0));
#pragma unroll
    for (int c = 0; c < NEQ / 2; ++c) {
      const float2 av = a[c];
      const double2 xx = xv[c];
      acc = fma((double)av.x, xx.x, acc);
      acc = fma((double)av.y, xx.y, acc);
    }
  }
  mbar_wait(bar, 0);
  if (!live) return;
  const int64_t bd = blkmap[(int64_t)BS * i];
  const float* __restrict__ a = sm + (b0 - i - s0) * PKF + base;
  for (int64_t b = b0; b < b1; ++b) {
    if (b == bd) continue;
    const double* __restrict__ xj = xs + NEQ * (b - B0);
    if (n == 8) {
      const float4* __restrict__ a4 = reinterpret_cast<const float4*>(a);
      const double2* __restrict__ x2 = reinterpret_cast<const double2*>(xj);
#pragma unroll
      for (int c = 0; c < 2; ++c) {
        const float4 av = a4[c];
        const double2 xa = x2[2 * c], xb = x2[2 * c + 1];
        acc = fma((double)av.y, xa.y, fma((double)av.x, xa.x, acc));
        acc = fma((double)av.w, xb.y, fma((double)av.z, xb.x, acc));
      }
    } else {
      acc = fma((double)a[0], xj[c0], acc);
      acc = fma((double)a[1], xj[cs], acc);
      acc = fma((double)a[2], xj[cs + 1], acc);
      acc = fma((double)a[3], xj[cs + 2], acc);
      acc = fma((double)a[4], xj[cT], acc);
    }
    a += PKF;
  }
  y[NEQ * i + r] = acc;
}
// z = D v with D = [nc][18][18] in FP32 (the preconditioner's application in the mixed-precision solve)
__global__ void __launch_bounds__(SV_T) k_diag_spmv_f32(int64_t nc, const float* __restrict__ dv,
                                                       const double* __restrict__ x, double* __restrict__ y) {
  const int r = threadIdx.x % NEQ;
  const int64_t i = blockIdx.x * (int64_t)SV_CELLS + threadIdx.x / NEQ;
  if (i >= nc) return;
  const float2* __restrict__ a = reinterpret_cast<const float2*>(dv + i * BLK + r * NEQ);
  const double2* __restrict__ xv = reinterpret_cast<const double2*>(x + NEQ * i);
  double acc = 0.0;
#pragma unroll
  for (int c = 0; c < NEQ / 2; ++c) {
    const float2 av = a[c];
    const double2 xx = xv[c];
    acc = fma((double)av.x, xx.x, acc);
    acc = fma((double)av.y, xx.y, acc);
  }
  y[NEQ * i + r] = acc;
}
static int launch_packed_spmv_f32(const tfa_mesh* m, const float* dvals, const float* ovals, const double* x, double* y,
                                  cudaStream_t st) {
  if ((reinterpret_cast<uintptr_t>(dvals) | reinterpret_cast<uintptr_t>(ovals) | reinterpret_cast<uintptr_t>(x)) & 15)
    return set_error(TFA_EINVAL, "tfa_gmres_packed_f32: the FP32 arrays and x must be 16-byte aligned");
  const size_t smem = 16 + sizeof(double) * NEQ * SV_CELLS * (m->F + 1) + sizeof(float) * SV_CELLS * m->F * PKF;
  k_packed_spmv_f32<<<cdiv(m->nc, SV_CELLS), SV_T, smem, st>>>(m->nc, blk_stride(m->F), m->F + 1, m->bsr_rowptr.p, m->bsr_col.p,
                                                              m->blkmap.p, dvals, ovals, x, y);
  return 0;
}

// packed -> BSR: thread (block b, entry e) of the mesh's pattern
__global__ void k_packed_to_bsr(int64_t nc, int64_t nnzb, int BS, const int32_t* __restrict__ rowptr,
                                const int32_t* __restrict__ blkmap, const int32_t* __restrict__ row_of_block,
                                const double* __restrict__ dvals, const double* __restrict__ ovals,
                                double* __restrict__ vals) {
  const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (t >= nnzb * BLK) return;
  const int64_t b = t / BLK;
  const int e = (int)(t - b * BLK), r = e / NEQ, c = e - NEQ * r;
  const int64_t i = row_of_block[b], bd = blkmap[(int64_t)BS * i];
  if (b == bd) { vals[t] = dvals[i * BLK + e]; return; }
  const int64_t slot = b - i - (b > bd ? 1 : 0);
  int base, n, c0, cs, cT;
  packed_row(r, base, n, c0, cs, cT);
  int cc = -1;   // position of column c inside the row's group, -1 outside it
  if (n == 8) cc = c < 8 ? c : -1;
  else cc = c == c0 ? 0 : (c == cT ? 4 : (c >= cs && c < cs + 3 ? 1 + c - cs : -1));
  vals[t] = cc >= 0 ? ovals[slot * TFA_PACKED_BLOCK + base + cc] : 0.0;
}
__global__ void k_row_of_block(int64_t nc, const int32_t* __restrict__ rowptr, int32_t* __restrict__ row_of_block) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= nc) return;
  for (int32_t b = rowptr[i]; b < rowptr[i + 1]; ++b) row_of_block[b] = (int32_t)i;
}

// ------------------------------------------------------------------------------------------------
// Inverse of each diagonal block: Gauss-Jordan with partial pivoting, FIVE blocks per warp.  A group of six lanes
// owns one block, lane r of the group keeping rows 3r..3r+2 in registers (54 doubles); rows are never moved: the
// pivot of step k is the largest |a[R][k]| among the rows not yet used, p_k, found by three shuffle rotations
// inside the group, and its row reaches the group through 144 bytes of shared memory.  Every value a lane
// receives feeds three FMAs, and one broadcast load serves five blocks: 11 shared-memory wavefronts and 11 FP64
// instructions per block and step, against 36 and 18 for the one-warp-per-block version before it
// (3.4 ms at 1M cells, its shared-memory data pipe 67 % busy: profiles/r1_ncu_full_block_jacobi_c4b.md).
// The blocks come in by TMA (one bulk load of 2592 B each) and go out the same way.  With P the permutation
// (PA)[k] = A[p_k], the in-place result S = (PA)^-1 sits as row k in the lane that owned p_k and
// A^-1[k][p_c] = S[k][c]; it is put in order in the shared-memory buffer the block arrived in.
// ------------------------------------------------------------------------------------------------
constexpr int BJ_WARPS = 4, BJ_G = 5, BJ_L = 6, BJ_R = 3;
// 1/d for a normal d: the hardware's 20-bit seed and two Newton steps (the pivot is never zero, subnormal or not
// finite: those end the inversion before this is reached)
__device__ __forceinline__ void bj_put_row(double2* __restrict__ dst, const double (&row)[NEQ]) {
#pragma unroll
  for (int c = 0; c < NEQ; c += 2) dst[c / 2] = make_double2(row[c], row[c + 1]);
}
__device__ __forceinline__ double bj_rcp(double d) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(d));
  double e = fma(-d, y, 1.0);
  y = fma(y, e, y);
  e = fma(-d, y, 1.0);
  return fma(y, e, y);
}
constexpr size_t BJ_SMEM = sizeof(double) * BJ_WARPS * (BJ_G * BLK + 2 * BJ_G * NEQ) + sizeof(uint64_t) * BJ_WARPS;
__global__ void __launch_bounds__(32 * BJ_WARPS, 3) k_block_jacobi(int64_t nc, const int32_t* __restrict__ blkmap, int BS,
                                                               const double* __restrict__ vals, int64_t nblk,
                                                               double* __restrict__ dinv, int32_t* __restrict__ flags) {
  extern __shared__ __align__(128) unsigned char bj_raw[];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  double(*buf)[BLK] = reinterpret_cast<double(*)[BLK]>(bj_raw) + w * BJ_G;
  // pivot rows: [2][BJ_G][18] doubles per warp (144 bytes apart: the five owners' 16-byte stores fall in distinct banks)
  double* const prows = reinterpret_cast<double*>(bj_raw) + BJ_WARPS * BJ_G * BLK + w * 2 * BJ_G * NEQ;
  uint64_t* bar = reinterpret_cast<uint64_t*>(bj_raw + sizeof(double) * BJ_WARPS * (BJ_G * BLK + 2 * BJ_G * NEQ)) + w;
  const int64_t i0 = (blockIdx.x * (int64_t)BJ_WARPS + w) * BJ_G;
  // no early return: a warp past the end runs with nb = 0 (the compiler must see all 32 lanes reach the shuffles)
  const int nb = (int)max((int64_t)0, min((int64_t)BJ_G, nc - i0));
  if (lane == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    mbar_arrive_expect_tx(bar, (uint32_t)(nb * BLK * sizeof(double)));
  }
  __syncwarp();
  // the diagonal block of row i (every row of the mesh's pattern has one); blkmap == NULL: vals is the packed
  // Jacobian's array of diagonal blocks
  if (lane < nb) {
    const int64_t i = i0 + lane, bd = blkmap ? (int64_t)blkmap[(int64_t)BS * i] : i;
    TFA_BOUND(flags, bd >= 0 && bd < nblk);
    bulk_load(buf[lane], vals + bd * BLK, (uint32_t)(BLK * sizeof(double)), bar);
  }
  const int g = lane / BJ_L, r = lane - BJ_L * g;
  const bool have = g < nb;                                     // lanes 30, 31 and the groups past the end idle
  const int gb = min(g, BJ_G - 1);                              // lanes 30, 31 read (never write) the last buffer
  const int gl0 = BJ_L * g;                                     // the group's first lane; its rotations by 1 and 2
  const int rot1 = g < BJ_G ? gl0 + (r + 1) % BJ_L : lane, rot2 = g < BJ_G ? gl0 + (r + 2) % BJ_L : lane;
  double a[BJ_R][NEQ];
  mbar_wait(bar, 0);
#pragma unroll
  for (int s = 0; s < BJ_R; ++s)
#pragma unroll
    for (int c = 0; c < NEQ; c += 2) {
      const double2 t = have ? *reinterpret_cast<const double2*>(&buf[g][(BJ_R * r + s) * NEQ + c]) : make_double2(0.0, 0.0);
      a[s][c] = t.x;
      a[s][c + 1] = t.y;
    }
  bool used[BJ_R] = {false, false, false}, singular = false;
  int myk[BJ_R] = {0, 0, 0};
  double scale[BJ_R] = {1.0, 1.0, 1.0};
  unsigned pk[3] = {0u, 0u, 0u};   // p_k, five bits each, six to a word
#pragma unroll
  for (int k = 0; k < NEQ; ++k) {
    // pivot: the largest |a[R][k]| over the rows not used yet, compared on the high word without its last five
    // bits (exponent and 15 mantissa bits: any entry within 2^-15 of the largest serves partial pivoting equally
    // well); those five bits carry 31 - R, so that ties go to the smallest R and one maximum over the group's
    // six lanes (three rotations by shuffle; a masked __reduce_max_sync runs once per group, six times slower)
    // gives the row as well.  NaN / Inf sort above every finite number and end the inversion.
    unsigned lkey = 0u;
#pragma unroll
    for (int s = 0; s < BJ_R; ++s) {
      const unsigned key = ((unsigned)__double2hiint(a[s][k]) & 0x7fffffe0u) | (unsigned)(31 - BJ_R * r - s);
      lkey = max(lkey, used[s] ? 0u : key);
    }
    lkey = max(lkey, __shfl_sync(0xffffffffu, lkey, rot1));
    lkey = max(lkey, __shfl_sync(0xffffffffu, lkey, rot2));
    const unsigned mx = max(lkey, __shfl_sync(0xffffffffu, lkey, rot2));
    if (mx < 32u || mx >= 0x7ff00000u) singular = true;   // group-uniform: zero / subnormal / not finite
    const int win = min(31 - (int)(mx & 31u), NEQ - 1);
    const int owner = gl0 + win / BJ_R, slot = win - BJ_R * (win / BJ_R);
    pk[k / 6] |= (unsigned)win << (5 * (k % 6));
    // rows other than the pivot row: a[c] <- a[c] + m t[c] with m = -a[k]/t[k], and column k becomes the inverse's,
    // m.  The pivot row is NOT divided by its pivot now: every later step acts linearly on it, so the factor
    // 1/t[k] is kept in `scale` and applied once at the end (its column k holds 1 until then).
    // the pivot row goes through 144 bytes of shared memory, double-buffered: its owner stores whichever of its
    // three rows it is -- the only place the dynamic row slot costs anything -- and the six lanes read it back as
    // broadcasts, one __syncwarp per step
    double2* __restrict__ prow = reinterpret_cast<double2*>(prows + ((k & 1) * BJ_G + gb) * NEQ);
    if (have && lane == owner) {
      if (slot == 0) bj_put_row(prow, a[0]);
      else if (slot == 1) bj_put_row(prow, a[1]);
      else bj_put_row(prow, a[2]);
    }
    __syncwarp();
    const double2 tkk = prow[k / 2];
    const double ip = bj_rcp(k & 1 ? tkk.y : tkk.x);
    double m[BJ_R];
#pragma unroll
    for (int s = 0; s < BJ_R; ++s) {
      const bool mine = BJ_R * r + s == win;
      m[s] = mine ? 0.0 : -(a[s][k] * ip);
      if (mine) {
        used[s] = true;
        myk[s] = k;
        scale[s] = ip;
      }
    }
#pragma unroll
    for (int c = 0; c < NEQ; c += 2) {
      const double2 t = prow[c / 2];
#pragma unroll
      for (int s = 0; s < BJ_R; ++s) {
        if (c != k) a[s][c] = fma(m[s], t.x, a[s][c]);
        if (c + 1 != k) a[s][c + 1] = fma(m[s], t.y, a[s][c + 1]);
      }
    }
#pragma unroll
    for (int s = 0; s < BJ_R; ++s) a[s][k] = (used[s] && myk[s] == k) ? 1.0 : m[s];
  }
  __syncwarp();
  if (have) {
#pragma unroll
    for (int s = 0; s < BJ_R; ++s)
#pragma unroll
      for (int c = 0; c < NEQ; ++c)
        buf[g][myk[s] * NEQ + (int)((pk[c / 6] >> (5 * (c % 6))) & 31u)] = scale[s] * a[s][c];
    if (singular) {   // the block's inverse is reported as zeros, and counted
      for (int e = r; e < BLK; e += BJ_L) buf[g][e] = 0.0;
      if (r == 0) atomicAdd(flags + 1, 1);
    }
  }
  fence_async_smem();
  __syncwarp();
  if (lane < nb) {
    bulk_store(dinv + (i0 + lane) * BLK, buf[lane], (uint32_t)(BLK * sizeof(double)));
    bulk_commit();
    bulk_wait_read();
  }
}
static int launch_block_jacobi(int64_t nc, const int32_t* blkmap, int BS, const double* vals, int64_t nblk,
                               double* dinv, int32_t* flags, cudaStream_t st) {
  if ((reinterpret_cast<uintptr_t>(vals) | reinterpret_cast<uintptr_t>(dinv)) & 15)
    return set_error(TFA_EINVAL, "tfa_block_jacobi: the block arrays must be 16-byte aligned");
  // per launch: the attribute belongs to the function on the CURRENT device, and the call is cheap
  TFA_CUDA(cudaFuncSetAttribute(k_block_jacobi, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)BJ_SMEM));
  k_block_jacobi<<<cdiv(nc, BJ_WARPS * BJ_G), 32 * BJ_WARPS, BJ_SMEM, st>>>(nc, blkmap, BS, vals, nblk, dinv, flags);
  return 0;
}

// ------------------------------------------------------------------------------------------------
// Vector kernels of GMRES.  Reductions are two-pass and deterministic: pass 1 writes per-CTA partial sums,
// pass 2 (one CTA) adds them in a fixed order.
// ------------------------------------------------------------------------------------------------
constexpr int RED_T = 256, RED_B = 592;

// part[b][j] = sum over the CTA's share of V_j . w, j < k  (V_j = V + j * ld); with `self`, entry k is w . w (the
// norm the Gram-Schmidt pass starts from, taken in the same pass over w).  Eight products per pass over w,
// 16-byte loads (n and ld are multiples of 18, hence even; the arrays are 16-byte aligned), the eight streams of a
// thread in flight together.
__global__ void __launch_bounds__(RED_T) k_dots(int64_t n, int k, const double* __restrict__ V, int64_t ld,
                                               const double* __restrict__ w, double* __restrict__ part, bool self) {
  __shared__ double sm[RED_T / 32];
  const int64_t n2 = n >> 1;
  const double2* __restrict__ w2 = reinterpret_cast<const double2*>(w);
  // caller-owned vectors need not be 16-byte aligned: then one element at a time
  const bool vec = !((reinterpret_cast<uintptr_t>(V) | reinterpret_cast<uintptr_t>(w)) & 15) && !(n & 1) && !(ld & 1);
  const int kk = k + (self ? 1 : 0);
  for (int j0 = 0; j0 < kk; j0 += 8) {
    double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    const int kj = min(8, kk - j0);
    const double* vp[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) vp[q] = j0 + q < k ? V + (int64_t)(j0 + q) * ld : w;
    if (!vec) {
      for (int64_t e = blockIdx.x * (int64_t)RED_T + threadIdx.x; e < n; e += (int64_t)RED_T * gridDim.x) {
        const double we = w[e];
#pragma unroll
        for (int q = 0; q < 8; ++q)
          if (q < kj) acc[q] = fma(vp[q][e], we, acc[q]);
      }
    } else if (kj == 8) {
      for (int64_t e = blockIdx.x * (int64_t)RED_T + threadIdx.x; e < n2; e += (int64_t)RED_T * gridDim.x) {
        const double2 we = w2[e];
        double2 v[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) v[q] = reinterpret_cast<const double2*>(vp[q])[e];
#pragma unroll
        for (int q = 0; q < 8; ++q) acc[q] = fma(v[q].y, we.y, fma(v[q].x, we.x, acc[q]));
      }
    } else {
      for (int64_t e = blockIdx.x * (int64_t)RED_T + threadIdx.x; e < n2; e += (int64_t)RED_T * gridDim.x) {
        const double2 we = w2[e];
#pragma unroll
        for (int q = 0; q < 8; ++q)
          if (q < kj) {
            const double2 v = reinterpret_cast<const double2*>(vp[q])[e];
            acc[q] = fma(v.y, we.y, fma(v.x, we.x, acc[q]));
          }
      }
    }
    for (int q = 0; q < kj; ++q) {
      double v = acc[q];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
      if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
      __syncthreads();
      if (threadIdx.x == 0) {
        double s = 0.0;
        for (int t = 0; t < RED_T / 32; ++t) s += sm[t];
        part[(int64_t)blockIdx.x * MAXK + j0 + q] = s;
      }
      __syncthreads();
    }
  }
}
// one warp per dot product: lane l adds the partial sums l, l + 32, ... in order, then a fixed shuffle tree
__global__ void __launch_bounds__(32) k_dots_final(int nblocks, const double* __restrict__ part,
                                                   double* __restrict__ out) {
  const int j = blockIdx.x;
  double s = 0.0;
  for (int b = threadIdx.x; b < nblocks; b += 32) s += part[(int64_t)b * MAXK + j];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (threadIdx.x == 0) out[j] = s;
}
// w -= sum_j h[j] V_j   (16-byte accesses; four basis vectors in flight at a time).  With `part` the CTA's share of
// the NEW w . w goes to part[b][0] (the norm after the Gram-Schmidt pass, from the values just computed).
__global__ void __launch_bounds__(RED_T) k_sub_combination(int64_t n, int k, const double* __restrict__ V, int64_t ld,
                                                          const double* __restrict__ h, double* __restrict__ w,
                                                          double* __restrict__ part) {
  __shared__ double hs[MAXK];
  __shared__ double sm[RED_T / 32];
  if (threadIdx.x < k) hs[threadIdx.x] = h[threadIdx.x];
  __syncthreads();
  const int64_t n2 = n >> 1, ld2 = ld >> 1;
  double2* __restrict__ w2 = reinterpret_cast<double2*>(w);
  const double2* __restrict__ V2 = reinterpret_cast<const double2*>(V);
  double nrm = 0.0;
  if (((reinterpret_cast<uintptr_t>(V) | reinterpret_cast<uintptr_t>(w)) & 15) || (n & 1) || (ld & 1)) {
    for (int64_t e = blockIdx.x * (int64_t)RED_T + threadIdx.x; e < n; e += (int64_t)RED_T * gridDim.x) {
      double v = w[e];
      for (int j = 0; j < k; ++j) v = fma(-hs[j], V[j * ld + e], v);
      w[e] = v;
      nrm = fma(v, v, nrm);
    }
  } else {
    for (int64_t e = blockIdx.x * (int64_t)RED_T + threadIdx.x; e < n2; e += (int64_t)RED_T * gridDim.x) {
      double2 v = w2[e];
      int j = 0;
      for (; j + 4 <= k; j += 4) {
        double2 t[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) t[q] = V2[(int64_t)(j + q) * ld2 + e];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          v.x = fma(-hs[j + q], t[q].x, v.x);
          v.y = fma(-hs[j + q], t[q].y, v.y);
        }
      }
      for (; j < k; ++j) {
        const double2 t = V2[(int64_t)j * ld2 + e];
        v.x = fma(-hs[j], t.x, v.x);
        v.y = fma(-hs[j], t.y, v.y);
      }
      w2[e] = v;
      nrm = fma(v.y, v.y, fma(v.x, v.x, nrm));
    }
  }
  if (!part) return;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) nrm += __shfl_xor_sync(0xffffffffu, nrm, o);
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = nrm;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int q = 0; q < RED_T / 32; ++q) t += sm[q];
    part[(int64_t)blockIdx.x * MAXK] = t;
  }
}
// ---- the same three kernels for a Krylov basis stored in FP32 (mixed-precision solve; w, the sums and the
// coefficients stay FP64).  Basis vectors are ld floats apart, ld a multiple of 4: 16-byte loads of four entries;
// n = 18 n_cells is even but need not be a multiple of 4: the last pair is handled by one thread. ----
__device__ __forceinline__ void block_sum_to(double v, double* sm, double* dst) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int q = 0; q < RED_T / 32; ++q) t += sm[q];
    *dst = t;
  }
  __syncthreads();
}
// v = fl32(a x): the new basis vector, and the same values in FP64 (what the preconditioner reads next)
__global__ void __launch_bounds__(RED_T) k_scale_f32(int64_t n, double a, const double* __restrict__ x,
                                                    float* __restrict__ v32, double* __restrict__ v64) {
  const int64_t n2 = n >> 1;
  const double2* __restrict__ x2 = reinterpret_cast<const double2*>(x);
  float2* __restrict__ o32 = reinterpret_cast<float2*>(v32);
  double2* __restrict__ o64 = reinterpret_cast<double2*>(v64);
  for (int64_t e = blockIdx.x * (int64_t)RED_T + threadIdx.x; e < n2; e += (int64_t)RED_T * gridDim.x) {
    const double2 t = x2[e];
    const float2 f = make_float2((float)(a * t.x), (float)(a * t.y));
    o32[e] = f;
    o64[e] = make_double2((double)f.x, (double)f.y);
  }
}
// part[b][j] = V_j . w for j < k, part[b][k] = w . w
__global__ void __launch_bounds__(RED_T) k_dots_f32(int64_t n, int k, const float* __restrict__ V, int64_t ld,
                                                   const double* __restrict__ w, double* __restrict__ part) {
  __shared__ double sm[RED_T / 32];
  const int64_t n4 = n >> 2, ld4 = ld >> 2;
  const double2* __restrict__ w2 = reinterpret_cast<const double2*>(w);
  const float4* __restrict__ V4 = reinterpret_cast<const float4*>(V);
  const bool tail = (n & 3) && blockIdx.x == 0 && threadIdx.x == 0;   // elements 4 n4, 4 n4 + 1
  for (int j0 = 0; j0 < k || j0 == 0; j0 += 8) {
    double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0}, self = 0.0;
    const int kj = min(8, k - j0);
    const float4* __restrict__ Vb = V4 + (int64_t)j0 * ld4;
    for (int64_t e = blockIdx.x * (int64_t)RED_T + threadIdx.x; e < n4; e += (int64_t)RED_T * gridDim.x) {
      const double2 wa = w2[2 * e], wb = w2[2 * e + 1];
      float4 v[8];
#pragma unroll
      for (int q = 0; q < 8; ++q)
        if (q < kj) v[q] = Vb[q * ld4 + e];
#pragma unroll
      for (int q = 0; q < 8; ++q)
        if (q < kj)
          acc[q] = fma((double)v[q].w, wb.y, fma((double)v[q].z, wb.x, fma((double)v[q].y, wa.y, fma((double)v[q].x, wa.x, acc[q]))));
      if (j0 == 0) self = fma(wb.y, wb.y, fma(wb.x, wb.x, fma(wa.y, wa.y, fma(wa.x, wa.x, self))));
    }
    if (tail) {
      const double2 wa = w2[2 * n4];
      for (int q = 0; q < kj; ++q) {
        const float* vq = V + (int64_t)(j0 + q) * ld + 4 * n4;
        acc[q] = fma((double)vq[1], wa.y, fma((double)vq[0], wa.x, acc[q]));
      }
      if (j0 == 0) self = fma(wa.y, wa.y, fma(wa.x, wa.x, self));
    }
    for (int q = 0; q < kj; ++q) block_sum_to(acc[q], sm, part + (int64_t)blockIdx.x * MAXK + j0 + q);
    if (j0 == 0) block_sum_to(self, sm, part + (int64_t)blockIdx.x * MAXK + k);
  }
}
// w -= sum_j h[j] V_j; with `part`, part[b][0] = the CTA's share of the new w . w
__global__ void __launch_bounds__(RED_T) k_sub_combination_f32(int64_t n, int k, const float* __restrict__ V, int64_t ld,
                                                              const double* __restrict__ h, double* __restrict__ w,
                                                              double* __restrict__ part) {
  __shared__ double hs[MAXK];
  __shared__ double sm[RED_T / 32];
  if (threadIdx.x < k) hs[threadIdx.x] = h[threadIdx.x];
  __syncthreads();
  const int64_t n4 = n >> 2, ld4 = ld >> 2;
  double2* __restrict__ w2 = reinterpret_cast<double2*>(w);
  const float4* __restrict__ V4 = reinterpret_cast<const float4*>(V);
  double nrm = 0.0;
  for (int64_t e = blockIdx.x * (int64_t)RED_T + threadIdx.x; e < n4; e += (int64_t)RED_T * gridDim.x) {
    double2 a = w2[2 * e], b = w2[2 * e + 1];
    int j = 0;
    for (; j + 4 <= k; j += 4) {
      float4 t[4];
#pragma unroll
      for (int q = 0; q < 4; ++q) t[q] = V4[(int64_t)(j + q) * ld4 + e];
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        a.x = fma(-hs[j + q], (double)t[q].x, a.x);
        a.y = fma(-hs[j + q], (double)t[q].y, a.y);
        b.x = fma(-hs[j + q], (double)t[q].z, b.x);
        b.y = fma(-hs[j + q], (double)t[q].w, b.y);
      }
    }
    for (; j < k; ++j) {
      const float4 t = V4[(int64_t)j * ld4 + e];
      a.x = fma(-hs[j], (double)t.x, a.x);
      a.y = fma(-hs[j], (double)t.y, a.y);
      b.x = fma(-hs[j], (double)t.z, b.x);
      b.y = fma(-hs[j], (double)t.w, b.y);
    }
    w2[2 * e] = a;
    w2[2 * e + 1] = b;
    nrm = fma(b.y, b.y, fma(b.x, b.x, fma(a.y, a.y, fma(a.x, a.x, nrm))));
  }
  if ((n & 3) && blockIdx.x == 0 && threadIdx.x == 0) {
    double2 a = w2[2 * n4];
    for (int j = 0; j < k; ++j) {
      const float* vq = V + (int64_t)j * ld + 4 * n4;
      a.x = fma(-hs[j], (double)vq[0], a.x);
      a.y = fma(-hs[j], (double)vq[1], a.y);
    }
    w2[2 * n4] = a;
    nrm = fma(a.y, a.y, fma(a.x, a.x, nrm));
  }
  if (part) block_sum_to(nrm, sm, part + (int64_t)blockIdx.x * MAXK);
}
// out = a * x + c * y   (y may be null with c = 0)
__global__ void __launch_bounds__(RED_T) k_axpby(int64_t n, double a, const double* __restrict__ x, double c,
                                                const double* __restrict__ y, double* __restrict__ out) {
  for (int64_t e = blockIdx.x * (int64_t)RED_T + threadIdx.x; e < n; e += (int64_t)RED_T * gridDim.x)
    out[e] = y ? fma(a, x[e], c * y[e]) : a * x[e];
}


namespace {

struct Gm {
  const tfa_mesh* m;
  const double *vals, *dinv;
  const double* vals_o;   // non-null: (vals, vals_o) is the packed Jacobian
  int64_t n;
  cudaStream_t st;
  double *part, *out;   // reduction scratch (device)
  double host[MAXK];
  std::function<int(const double*, double*)> op;   // y = A x when the matrix is not assembled (JFNK)
  // mixed precision: the operator of the Krylov cycle (FP32 matrix) -- the residual at a restart still uses spmv --
  // and the preconditioner's application (FP32 blocks)
  std::function<int(const double*, double*)> op_inner;
  std::function<void(const double*, double*)> pre;

  int spmv_inner(const double* x, double* y) const { return op_inner ? op_inner(x, y) : spmv(x, y); }
  int spmv(const double* x, double* y) const {
    if (op) return op(x, y);
    if (vals_o)
      return launch_packed_spmv(m, vals, vals_o, x, y, st);
    else
      k_bsr_spmv<false><<<cdiv(m->nc, SV_CELLS), SV_T, 0, st>>>(m->nc, m->bsr_rowptr.p, m->bsr_col.p, vals, x, y);
    return 0;
  }
  // z = M^-1 v (block-diagonal product), or a copy without preconditioner
  void precond(const double* v, double* z) const {
    if (pre) pre(v, z);
    else if (dinv) k_bsr_spmv<true><<<cdiv(m->nc, SV_CELLS), SV_T, 0, st>>>(m->nc, nullptr, nullptr, dinv, v, z);
    else k_axpby<<<RED_B, RED_T, 0, st>>>(n, 1.0, v, 0.0, nullptr, z);
  }
  // host[j] = V_j . w for j < k (synchronises)
  int dots(int k, const double* V, int64_t ld, const double* w) {
    k_dots<<<RED_B, RED_T, 0, st>>>(n, k, V, ld, w, part, false);
    k_dots_final<<<k, 32, 0, st>>>(RED_B, part, out);
    TFA_CUDA(cudaMemcpyAsync(host, out, sizeof(double) * k, cudaMemcpyDeviceToHost, st));
    TFA_CUDA(cudaStreamSynchronize(st));
    return 0;
  }
};

}  // namespace
}  // namespace tfa

using namespace tfa;

static int gmres_core(tfa_ctx* ctx, const tfa_mesh* m, const double* bsr_vals, const double* dinv,
                      std::function<int(const double*, double*)> op, const double* b, double* x, int restart,
                      int max_iters, double rtol, double* info, void* stream, const double* offd_vals = nullptr,
                      std::function<int(const double*, double*)> op_inner = nullptr,
                      std::function<void(const double*, double*)> pre = nullptr, double inner_floor = 0.0,
                      bool basis32 = false) {
  if (restart < 1 || restart > MAXK - 2 || max_iters < 0 || !(rtol >= 0.0))
    return set_error(TFA_EINVAL, "tfa_gmres: restart must be in 1..62, max_iters >= 0, rtol >= 0");
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t n = (int64_t)NEQ * m->nc;
  const int mk = restart;
  const int64_t ld32 = (n + 3) & ~(int64_t)3;   // FP32 basis: vectors this many floats apart
  const int64_t off32 = (((int64_t)(mk + 1) * ld32 + 1) / 2 + 1) & ~(int64_t)1;   // its size in doubles, even
  const int64_t need = std::max((int64_t)(mk + 3) * n, basis32 ? off32 + 3 * n : (int64_t)0);
  if (ctx->krylov.n < need) TFA_CUDA(ctx->krylov.alloc(need));
  if (ctx->red.n < (int64_t)RED_B * MAXK + MAXK) TFA_CUDA(ctx->red.alloc((int64_t)RED_B * MAXK + MAXK));
  double* V = ctx->krylov.p;              // V_0 .. V_mk
  double* w = V + (int64_t)(mk + 1) * n;  // work vector
  double* z = w + n;                      // preconditioned vector
  // mixed precision: the basis in FP32 (vectors ld32 floats apart), the newest basis vector also in FP64 (vcur)
  float* V32 = reinterpret_cast<float*>(ctx->krylov.p);
  double* vcur = nullptr;
  if (basis32) {
    w = ctx->krylov.p + off32;
    z = w + n;
    vcur = z + n;
  }
  Gm G{m, bsr_vals, dinv, offd_vals, n, st, ctx->red.p, ctx->red.p + (int64_t)RED_B * MAXK, {}, op, op_inner, pre};

  TFA_TRY(G.dots(1, b, n, b));
  const double bnorm = std::sqrt(G.host[0]);
  if (bnorm == 0.0) {   // b = 0: x = 0
    TFA_CUDA(cudaMemsetAsync(x, 0, sizeof(double) * n, st));
    return 0;
  }
  int iters = 0;
  std::vector<double> H((size_t)(mk + 1) * mk), cs(mk), sn(mk), g(mk + 1), yv(mk);
  double rel = 0.0;
  for (;;) {
    // r = b - A x  (true residual at every restart)
    TFA_TRY(G.spmv(x, w));
    k_axpby<<<RED_B, RED_T, 0, st>>>(n, 1.0, b, -1.0, w, w);
    TFA_TRY(G.dots(1, w, n, w));
    const double beta = std::sqrt(G.host[0]);
    rel = beta / bnorm;
    info[0] = (double)iters;
    info[1] = rel;
    // a non-finite residual (NaN / Inf in the matrix, the preconditioner or b): x holds the last iterate
    if (!std::isfinite(beta)) return set_error(TFA_ESINGULAR, "tfa_gmres: the residual norm is not finite");
    if (rel <= rtol || iters >= max_iters) break;
    if (basis32) k_scale_f32<<<RED_B, RED_T, 0, st>>>(n, 1.0 / beta, w, V32, vcur);
    else k_axpby<<<RED_B, RED_T, 0, st>>>(n, 1.0 / beta, w, 0.0, nullptr, V);
    std::fill(g.begin(), g.end(), 0.0);
    g[0] = beta;
    int k = 0;
    for (; k < mk && iters < max_iters; ++k, ++iters) {
      G.precond(basis32 ? vcur : V + (int64_t)k * n, z);
      TFA_TRY(G.spmv_inner(z, w));
      // classical Gram-Schmidt (all projections from one pass over the basis), repeated when it cancelled more
      // than a factor 10 of the vector (the Daniel-Gragg-Kaufman-Stewart test with eta = 0.1: the loss of
      // orthogonality of a single pass grows like eps / eta^2, and on the preconditioned systems of the method a
      // pass keeps 0.3-0.6 of the norm).  One pass = two kernels and ONE synchronisation: the projections stay on
      // the device between them, the norm before comes out of the first (entry k + 1), the norm after out of the
      // second (entry k + 2).
      double* h = &H[(size_t)k * (mk + 1)];
      for (int j = 0; j <= k + 1; ++j) h[j] = 0.0;
      double hk1 = 0.0;
      for (int pass = 0; pass < 2; ++pass) {
        if (basis32) k_dots_f32<<<RED_B, RED_T, 0, st>>>(n, k + 1, V32, ld32, w, G.part);
        else k_dots<<<RED_B, RED_T, 0, st>>>(n, k + 1, V, n, w, G.part, true);
        k_dots_final<<<k + 2, 32, 0, st>>>(RED_B, G.part, G.out);
        if (basis32) k_sub_combination_f32<<<RED_B, RED_T, 0, st>>>(n, k + 1, V32, ld32, G.out, w, G.part);
        else k_sub_combination<<<RED_B, RED_T, 0, st>>>(n, k + 1, V, n, G.out, w, G.part);
        k_dots_final<<<1, 32, 0, st>>>(RED_B, G.part, G.out + k + 2);
        TFA_CUDA(cudaMemcpyAsync(G.host, G.out, sizeof(double) * (k + 3), cudaMemcpyDeviceToHost, st));
        TFA_CUDA(cudaStreamSynchronize(st));
        for (int j = 0; j <= k; ++j) h[j] += G.host[j];
        const double before = std::sqrt(G.host[k + 1]);
        hk1 = std::sqrt(G.host[k + 2]);
        if (!(hk1 <= 0.1 * before)) break;   // also leaves on NaN
      }
      h[k + 1] = hk1;
      if (!std::isfinite(hk1)) return set_error(TFA_ESINGULAR, "tfa_gmres: a Krylov vector is not finite");
      if (hk1 > 0.0) {
        if (basis32) k_scale_f32<<<RED_B, RED_T, 0, st>>>(n, 1.0 / hk1, w, V32 + (int64_t)(k + 1) * ld32, vcur);
        else k_axpby<<<RED_B, RED_T, 0, st>>>(n, 1.0 / hk1, w, 0.0, nullptr, V + (int64_t)(k + 1) * n);
      }
      // Givens rotations on column k of the Hessenberg matrix
      for (int j = 0; j < k; ++j) {
        const double t = cs[j] * h[j] + sn[j] * h[j + 1];
        h[j + 1] = -sn[j] * h[j] + cs[j] * h[j + 1];
        h[j] = t;
      }
      const double den = std::hypot(h[k], h[k + 1]);
      // breakdown with a singular Hessenberg column (A M^-1 maps the Krylov space into itself without reaching
      // b): the least-squares problem has no unique solution; x keeps the previous cycle's iterate
      if (den == 0.0) return set_error(TFA_ESINGULAR, "tfa_gmres: breakdown on a singular operator");
      cs[k] = den > 0.0 ? h[k] / den : 1.0;
      sn[k] = den > 0.0 ? h[k + 1] / den : 0.0;
      h[k] = den;
      h[k + 1] = 0.0;
      g[k + 1] = -sn[k] * g[k];
      g[k] = cs[k] * g[k];
      // (mixed precision: a cycle ends once it has reduced ITS residual by inner_floor -- below that the FP32
      // operator's rounding, not the Krylov space, limits the true residual, which the restart recomputes in FP64)
      if (std::fabs(g[k + 1]) <= rtol * bnorm || hk1 == 0.0 || std::fabs(g[k + 1]) <= inner_floor * beta) {
        ++k;
        ++iters;
        break;
      }
    }
    // y = H^-1 g (upper triangular), u = sum_j y_j V_j, x += M^-1 u
    for (int i2 = k - 1; i2 >= 0; --i2) {
      double sacc = g[i2];
      for (int j = i2 + 1; j < k; ++j) sacc -= H[(size_t)j * (mk + 1) + i2] * yv[j];
      yv[i2] = sacc / H[(size_t)i2 * (mk + 1) + i2];
    }
    if (k > 0) {
      for (int j = 0; j < k; ++j) G.host[j] = -yv[j];
      TFA_CUDA(cudaMemcpyAsync(G.out, G.host, sizeof(double) * k, cudaMemcpyHostToDevice, st));
      TFA_CUDA(cudaMemsetAsync(w, 0, sizeof(double) * n, st));
      if (basis32) k_sub_combination_f32<<<RED_B, RED_T, 0, st>>>(n, k, V32, ld32, G.out, w, nullptr);
      else k_sub_combination<<<RED_B, RED_T, 0, st>>>(n, k, V, n, G.out, w, nullptr);   // w = sum_j y_j V_j
      TFA_CUDA(cudaStreamSynchronize(st));
      G.precond(w, z);
      k_axpby<<<RED_B, RED_T, 0, st>>>(n, 1.0, z, 1.0, x, x);
    }
  }
  TFA_CUDA(cudaGetLastError());
  info[0] = (double)iters;
  info[1] = rel;
  return 0;
}


extern "C" {

int tfa_bsr_spmv(const tfa_mesh* m, const double* bsr_vals, const double* x, double* y, void* stream) {
  if (!m) return set_error(TFA_EINVAL, "null argument");
  if (m->nc == 0) return 0;
  if (!bsr_vals || !x || !y) return set_error(TFA_EINVAL, "null argument");
  k_bsr_spmv<false><<<cdiv(m->nc, SV_CELLS), SV_T, 0, (cudaStream_t)stream>>>(m->nc, m->bsr_rowptr.p, m->bsr_col.p,
                                                                            bsr_vals, x, y);
  TFA_CUDA(cudaGetLastError());
  return 0;
}

int tfa_block_jacobi(tfa_ctx* ctx, const tfa_mesh* m, const double* bsr_vals, double* dinv, void* stream) {
  if (!ctx || !m) return set_error(TFA_EINVAL, "null argument");
  if (m->nc == 0) return 0;
  if (!bsr_vals || !dinv) return set_error(TFA_EINVAL, "null argument");
  cudaStream_t st = (cudaStream_t)stream;
  if (!ctx->flags.p) {
    TFA_CUDA(ctx->flags.alloc(4));
    TFA_CUDA(cudaMemsetAsync(ctx->flags.p, 0, 16, st));
  }
  TFA_TRY(launch_block_jacobi(m->nc, m->blkmap.p, blk_stride(m->F), bsr_vals, m->nnzb, dinv, ctx->flags.p, st));
  TFA_CUDA(cudaGetLastError());
  return 0;
}

int tfa_gmres(tfa_ctx* ctx, const tfa_mesh* m, const double* bsr_vals, const double* dinv, const double* b,
              double* x, int restart, int max_iters, double rtol, double* info, void* stream) {
  if (!ctx || !m || !info) return set_error(TFA_EINVAL, "null argument");
  info[0] = 0.0;
  info[1] = 0.0;
  if (m->nc == 0) return 0;
  if (!bsr_vals || !b || !x) return set_error(TFA_EINVAL, "null argument");
  return gmres_core(ctx, m, bsr_vals, dinv, nullptr, b, x, restart, max_iters, rtol, info, stream);
}

// ---- one implicit time step: the Newton sub-iterations of Eq. 14 (L120-128) around the entry points above ----
int tfa_implicit_step(tfa_ctx* ctx, const tfa_mesh* m, double* state, const double* state_n, const double* state_nm1,
                      double dt, double* rhs, double* bsr_vals, double* dinv, double* dP, int max_newton,
                      double newton_tol, int restart, int max_iters, double rtol, int matrix_free, double* info,
                      void* stream) {
  if (!ctx || !m || !info) return set_error(TFA_EINVAL, "null argument");
  for (int q = 0; q < 4; ++q) info[q] = 0.0;
  if (m->nc == 0) return 0;
  if (!state || !state_n || !state_nm1 || !rhs || !bsr_vals || !dinv || !dP) return set_error(TFA_EINVAL, "null argument");
  if (state == state_n || state == state_nm1) return set_error(TFA_EINVAL, "tfa_implicit_step: state must not alias P^n or P^{n-1}");
  if (max_newton < 1 || !(newton_tol >= 0.0)) return set_error(TFA_EINVAL, "tfa_implicit_step: max_newton >= 1, newton_tol >= 0");
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t n = (int64_t)NEQ * m->nc;
  if (ctx->red.n < (int64_t)RED_B * MAXK + MAXK) TFA_CUDA(ctx->red.alloc((int64_t)RED_B * MAXK + MAXK));
  double gm[2];
  if (matrix_free < 0 || matrix_free > 2) return set_error(TFA_EINVAL, "tfa_implicit_step: mode must be 0, 1 or 2");
  // mode 2: packed Jacobian inside the caller's value array (it always fits), FP32 copies in the context
  const int64_t n_offd = m->nnzb - m->nc;
  double *pk_d = bsr_vals, *pk_o = bsr_vals + m->nc * (int64_t)BLK;
  float *d32 = nullptr, *o32 = nullptr, *i32 = nullptr;
  if (matrix_free == 2) {
    const int64_t need = 2 * m->nc * (int64_t)BLK + n_offd * PKF;
    if (ctx->mixed.n < need) TFA_CUDA(ctx->mixed.alloc(need));
    d32 = ctx->mixed.p;
    o32 = d32 + m->nc * (int64_t)BLK;
    i32 = o32 + n_offd * PKF;
  }
  for (int it = 0; it < max_newton; ++it) {
    if (matrix_free == 2) {
      TFA_TRY(tfa_assemble_packed(ctx, m, state, state_n, state_nm1, dt, rhs, pk_d, pk_o, stream));
      TFA_TRY(tfa_block_jacobi_packed(ctx, m, pk_d, dinv, stream));
      TFA_TRY(tfa_packed_to_f32(m, pk_d, pk_o, d32, o32, stream));
      TFA_TRY(tfa_to_f32(dinv, i32, m->nc * (int64_t)BLK, stream));
    } else {
      TFA_TRY(tfa_assemble(ctx, m, state, state_n, state_nm1, dt, rhs, bsr_vals, stream));
      TFA_TRY(tfa_block_jacobi(ctx, m, bsr_vals, dinv, stream));
    }
    TFA_CUDA(cudaMemsetAsync(dP, 0, sizeof(double) * n, st));
    if (matrix_free == 2)
      TFA_TRY(tfa_gmres_packed_f32(ctx, m, pk_d, pk_o, d32, o32, i32, rhs, dP, restart, max_iters, rtol, gm, stream));
    else if (matrix_free)
      TFA_TRY(tfa_gmres_jfnk(ctx, m, state, state_n, state_nm1, dt, dinv, rhs, dP, restart, max_iters, rtol, gm, stream));
    else
      TFA_TRY(tfa_gmres(ctx, m, bsr_vals, dinv, rhs, dP, restart, max_iters, rtol, gm, stream));
    info[2] += gm[0];
    info[3] = gm[1];
    k_axpby<<<RED_B, RED_T, 0, st>>>(n, 1.0, dP, 1.0, state, state);   // P += dP
    Gm G{m, nullptr, nullptr, nullptr, n, st, ctx->red.p, ctx->red.p + (int64_t)RED_B * MAXK, {}, nullptr};
    TFA_TRY(G.dots(1, dP, n, dP));
    const double nd = std::sqrt(G.host[0]);
    TFA_TRY(G.dots(1, state, n, state));
    const double np = std::sqrt(G.host[0]);
    info[0] = it + 1;
    info[1] = nd / (1.0 + np);
    if (!std::isfinite(nd)) return set_error(TFA_ESINGULAR, "tfa_implicit_step: the Newton update is not finite");
    if (info[1] <= newton_tol) break;
  }
  TFA_CUDA(cudaGetLastError());
  return 0;
}

// ---- packed Jacobian (second option; include/tfa.h) ----
int tfa_packed_spmv(const tfa_mesh* m, const double* diag_vals, const double* offd_vals, const double* x, double* y,
                    void* stream) {
  if (!m) return set_error(TFA_EINVAL, "null argument");
  if (m->nc == 0) return 0;
  if (!diag_vals || !x || !y || (!offd_vals && m->nnzb > m->nc)) return set_error(TFA_EINVAL, "null argument");
  TFA_TRY(launch_packed_spmv(m, diag_vals, offd_vals, x, y, (cudaStream_t)stream));
  TFA_CUDA(cudaGetLastError());
  return 0;
}

int tfa_packed_to_bsr(const tfa_mesh* m, const double* diag_vals, const double* offd_vals, double* bsr_vals,
                      void* stream) {
  if (!m) return set_error(TFA_EINVAL, "null argument");
  if (m->nc == 0) return 0;
  if (!diag_vals || !bsr_vals || (!offd_vals && m->nnzb > m->nc)) return set_error(TFA_EINVAL, "null argument");
  cudaStream_t st = (cudaStream_t)stream;
  DevBuf<int32_t> rob;
  TFA_CUDA(rob.alloc(m->nnzb));
  k_row_of_block<<<cdiv(m->nc, 256), 256, 0, st>>>(m->nc, m->bsr_rowptr.p, rob.p);
  k_packed_to_bsr<<<cdiv(m->nnzb * BLK, 256), 256, 0, st>>>(m->nc, m->nnzb, blk_stride(m->F), m->bsr_rowptr.p,
                                                          m->blkmap.p, rob.p, diag_vals, offd_vals, bsr_vals);
  TFA_CUDA(cudaGetLastError());
  TFA_CUDA(cudaStreamSynchronize(st));   // the block-to-row table is a temporary
  return 0;
}

int tfa_block_jacobi_packed(tfa_ctx* ctx, const tfa_mesh* m, const double* diag_vals, double* dinv, void* stream) {
  if (!ctx || !m) return set_error(TFA_EINVAL, "null argument");
  if (m->nc == 0) return 0;
  if (!diag_vals || !dinv) return set_error(TFA_EINVAL, "null argument");
  cudaStream_t st = (cudaStream_t)stream;
  if (!ctx->flags.p) {
    TFA_CUDA(ctx->flags.alloc(4));
    TFA_CUDA(cudaMemsetAsync(ctx->flags.p, 0, 16, st));
  }
  TFA_TRY(launch_block_jacobi(m->nc, nullptr, 0, diag_vals, m->nc, dinv, ctx->flags.p, st));
  TFA_CUDA(cudaGetLastError());
  return 0;
}

int tfa_gmres_packed(tfa_ctx* ctx, const tfa_mesh* m, const double* diag_vals, const double* offd_vals,
                     const double* dinv, const double* b, double* x, int restart, int max_iters, double rtol,
                     double* info, void* stream) {
  if (!ctx || !m || !info) return set_error(TFA_EINVAL, "null argument");
  info[0] = 0.0;
  info[1] = 0.0;
  if (m->nc == 0) return 0;
  if (!diag_vals || !b || !x || (!offd_vals && m->nnzb > m->nc)) return set_error(TFA_EINVAL, "null argument");
  return gmres_core(ctx, m, diag_vals, dinv, nullptr, b, x, restart, max_iters, rtol, info, stream,
                    offd_vals ? offd_vals : diag_vals);
}

// ---- mixed precision on the packed Jacobian (include/tfa.h) ----
int tfa_to_f32(const double* src, float* dst, int64_t n, void* stream) {
  if (n < 0 || (n > 0 && (!src || !dst))) return set_error(TFA_EINVAL, "bad argument");
  if (n == 0) return 0;
  k_to_f32<<<1184, 256, 0, (cudaStream_t)stream>>>(n, src, dst);
  TFA_CUDA(cudaGetLastError());
  return 0;
}
int tfa_packed_to_f32(const tfa_mesh* m, const double* diag_vals, const double* offd_vals, float* diag32, float* offd32,
                      void* stream) {
  if (!m) return set_error(TFA_EINVAL, "null argument");
  if (m->nc == 0) return 0;
  const int64_t no = m->nnzb - m->nc;
  if (!diag_vals || !diag32 || (no > 0 && (!offd_vals || !offd32))) return set_error(TFA_EINVAL, "null argument");
  k_to_f32<<<1184, 256, 0, (cudaStream_t)stream>>>(m->nc * (int64_t)BLK, diag_vals, diag32);
  if (no > 0) k_offd_to_f32<<<1184, 256, 0, (cudaStream_t)stream>>>(no, offd_vals, offd32);
  TFA_CUDA(cudaGetLastError());
  return 0;
}
int tfa_gmres_packed_f32(tfa_ctx* ctx, const tfa_mesh* m, const double* diag_vals, const double* offd_vals,
                         const float* diag32, const float* offd32, const float* dinv32, const double* b, double* x,
                         int restart, int max_iters, double rtol, double* info, void* stream) {
  if (!ctx || !m || !info) return set_error(TFA_EINVAL, "null argument");
  info[0] = 0.0;
  info[1] = 0.0;
  if (m->nc == 0) return 0;
  const bool offd = m->nnzb > m->nc;
  if (!diag_vals || !diag32 || !b || !x || (offd && (!offd_vals || !offd32))) return set_error(TFA_EINVAL, "null argument");
  cudaStream_t st = (cudaStream_t)stream;
  auto inner = [=](const double* xin, double* yout) -> int {
    return launch_packed_spmv_f32(m, diag32, offd ? offd32 : diag32, xin, yout, st);
  };
  std::function<void(const double*, double*)> pre;
  if (dinv32)
    pre = [=](const double* v, double* z) { k_diag_spmv_f32<<<cdiv(m->nc, SV_CELLS), SV_T, 0, st>>>(m->nc, dinv32, v, z); };
  return gmres_core(ctx, m, diag_vals, nullptr, nullptr, b, x, restart, max_iters, rtol, info, stream,
                    offd ? offd_vals : diag_vals, inner, pre, 1e-5, true);
}

// ---- matrix-free operator (the paper's future work, L130) ----
static int jvp_core(tfa_ctx* ctx, const tfa_mesh* m, const double* state, const double* state_n,
                    const double* state_nm1, double dt, const double* rhs0, const double* v, double* out, double eps,
                    double rms_state, void* stream) {
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t n = (int64_t)NEQ * m->nc;
  if (ctx->jfnk.n < 2 * n) TFA_CUDA(ctx->jfnk.alloc(2 * n));
  if (ctx->red.n < (int64_t)RED_B * MAXK + MAXK) TFA_CUDA(ctx->red.alloc((int64_t)RED_B * MAXK + MAXK));
  double *Pp = ctx->jfnk.p, *rp = Pp + n;
  if (!(eps > 0.0)) {
    // eps = 1e-7 (1 + rms(P)) / rms(v)
    Gm G{m, nullptr, nullptr, nullptr, n, st, ctx->red.p, ctx->red.p + (int64_t)RED_B * MAXK, {}, nullptr};
    TFA_TRY(G.dots(1, v, n, v));
    const double rv = std::sqrt(G.host[0] / (double)n);
    if (rv == 0.0) {
      TFA_CUDA(cudaMemsetAsync(out, 0, sizeof(double) * n, st));
      return 0;
    }
    if (rms_state < 0.0) {
      TFA_TRY(G.dots(1, state, n, state));
      rms_state = std::sqrt(G.host[0] / (double)n);
    }
    eps = 1e-7 * (1.0 + rms_state) / rv;
  }
  k_axpby<<<RED_B, RED_T, 0, st>>>(n, eps, v, 1.0, state, Pp);                                  // P + eps v
  TFA_TRY(assemble_impl(ctx, m, Pp, state_n, state_nm1, dt, rp, nullptr, stream, false));   // rhs = -R~
  k_axpby<<<RED_B, RED_T, 0, st>>>(n, -1.0 / eps, rp, 1.0 / eps, rhs0, out);                    // (R~' - R~) / eps
  TFA_CUDA(cudaGetLastError());
  return 0;
}

int tfa_jvp(tfa_ctx* ctx, const tfa_mesh* m, const double* state, const double* state_n, const double* state_nm1,
            double dt, const double* v, double* out, double eps, void* stream) {
  if (!ctx || !m) return set_error(TFA_EINVAL, "null argument");
  if (m->nc == 0) return 0;
  if (!state || !state_n || !state_nm1 || !v || !out) return set_error(TFA_EINVAL, "null argument");
  const int64_t n = (int64_t)NEQ * m->nc;
  if (ctx->jfnk0.n < n) TFA_CUDA(ctx->jfnk0.alloc(n));
  TFA_TRY(assemble_impl(ctx, m, state, state_n, state_nm1, dt, ctx->jfnk0.p, nullptr, stream, false));
  return jvp_core(ctx, m, state, state_n, state_nm1, dt, ctx->jfnk0.p, v, out, eps, -1.0, stream);
}

int tfa_gmres_jfnk(tfa_ctx* ctx, const tfa_mesh* m, const double* state, const double* state_n,
                   const double* state_nm1, double dt, const double* dinv, const double* b, double* x, int restart,
                   int max_iters, double rtol, double* info, void* stream) {
  if (!ctx || !m || !info) return set_error(TFA_EINVAL, "null argument");
  info[0] = 0.0;
  info[1] = 0.0;
  if (m->nc == 0) return 0;
  if (!state || !state_n || !state_nm1 || !b || !x) return set_error(TFA_EINVAL, "null argument");
  if (!(dt > 0.0)) return set_error(TFA_EINVAL, "dt must be positive");
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t n = (int64_t)NEQ * m->nc;
  if (ctx->jfnk0.n < n) TFA_CUDA(ctx->jfnk0.alloc(n));
  if (ctx->red.n < (int64_t)RED_B * MAXK + MAXK) TFA_CUDA(ctx->red.alloc((int64_t)RED_B * MAXK + MAXK));
  // the base residual and the state's size, once per solve
  TFA_TRY(assemble_impl(ctx, m, state, state_n, state_nm1, dt, ctx->jfnk0.p, nullptr, stream, false));
  Gm G{m, nullptr, nullptr, nullptr, n, st, ctx->red.p, ctx->red.p + (int64_t)RED_B * MAXK, {}, nullptr};
  TFA_TRY(G.dots(1, state, n, state));
  const double rms_state = std::sqrt(G.host[0] / (double)n);
  auto op = [=](const double* xin, double* yout) -> int {
    return jvp_core(ctx, m, state, state_n, state_nm1, dt, ctx->jfnk0.p, xin, yout, 0.0, rms_state, stream);
  };
  return gmres_core(ctx, m, nullptr, dinv, op, b, x, restart, max_iters, rtol, info, stream);
}
}  // extern "C"
