// SIMT (CUDA-core, fp32 arithmetic) kernels of the Evoformer block, templated on the storage type of
// intermediates (float for the PF_F32 path; the 16-bit instantiations serve the parts of PF_BF16 that are
// not contractions).  Formulas: SURVEY.md Appendix A; readings R3-R7, R12.
#include "pf_internal.h"
#include "pf_device.cuh"

namespace pf {

// ---------------------------------------------------------------------------------------------
// LayerNorm over channels of fp32 residual rows (R4), optional transposed row gather.
// One warp per row, 128-bit loads, warp-shuffle reductions, two-pass variance.
// ---------------------------------------------------------------------------------------------
template <typename T, int NV>   // C = NV * 128
__global__ void __launch_bounds__(256) ln_rows_kernel(const float* __restrict__ x, T* __restrict__ y,
                                                      const float* __restrict__ gamma, const float* __restrict__ beta,
                                                      long rows, RowGeom g, int transposed) {
  const int C = NV * 128;
  long r = (long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (r >= rows) return;
  int lane = threadIdx.x & 31;
  long src = transposed ? transposed_row(r, g) : r;
  const float4* xp = reinterpret_cast<const float4*>(x + src * C);
  float4 v[NV];
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    v[i] = ld_nc_f4(xp + lane + 32 * i);
    s += v[i].x + v[i].y + v[i].z + v[i].w;
  }
  float mean = warp_sum(s) * (1.0f / C);
  float q = 0.f;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    float a = v[i].x - mean, b = v[i].y - mean, c = v[i].z - mean, d = v[i].w - mean;
    q += a * a + b * b + c * c + d * d;
  }
  float rstd = rsqrtf(warp_sum(q) * (1.0f / C) + 1e-5f);
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    int c4 = lane + 32 * i;
    float4 gm = __ldg(reinterpret_cast<const float4*>(gamma) + c4);
    float4 bt = __ldg(reinterpret_cast<const float4*>(beta) + c4);
    float4 o;
    o.x = (v[i].x - mean) * rstd * gm.x + bt.x;
    o.y = (v[i].y - mean) * rstd * gm.y + bt.y;
    o.z = (v[i].z - mean) * rstd * gm.z + bt.z;
    o.w = (v[i].w - mean) * rstd * gm.w + bt.w;
    store4(y + r * C + c4 * 4, o);
  }
}

template <typename T>
void launch_ln_rows(const float* x, T* y, const float* gamma, const float* beta, long rows, int C, RowGeom geom,
                    int transposed, cudaStream_t st) {
  int wpb = 8;
  unsigned grid = (unsigned)((rows + wpb - 1) / wpb);
  if (C == 128)
    ln_rows_kernel<T, 1><<<grid, wpb * 32, 0, st>>>(x, y, gamma, beta, rows, geom, transposed);
  else
    ln_rows_kernel<T, 2><<<grid, wpb * 32, 0, st>>>(x, y, gamma, beta, rows, geom, transposed);
}
template void launch_ln_rows<float>(const float*, float*, const float*, const float*, long, int, RowGeom, int, cudaStream_t);
template void launch_ln_rows<bf16>(const float*, bf16*, const float*, const float*, long, int, RowGeom, int, cudaStream_t);

// ---------------------------------------------------------------------------------------------
// Generic SIMT GEMM  acc[r,n] = sum_k A[r,k] W[k,n]  (+ second accumulator with W2 for gated pairs),
// 64x64 tile, 16-deep k-slices, 4x4 micro-tile per thread, shared epilogue (pf_device.cuh).
// ---------------------------------------------------------------------------------------------
template <typename T, bool DUAL>
__global__ void __launch_bounds__(256) gemm_simt_kernel(const T* __restrict__ A, int lda, const float* __restrict__ W,
                                                        const float* __restrict__ W2, int ldw, long R, int K, int Nout,
                                                        Epi epi) {
  __shared__ float As[16][64 + 4];
  __shared__ float Bs[16][64];
  __shared__ float Bs2[DUAL ? 16 : 1][64];
  int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  long r0 = (long)blockIdx.x * 64;
  int n0 = blockIdx.y * 64;
  float acc[4][4] = {}, acc2[4][4] = {};
  for (int k0 = 0; k0 < K; k0 += 16) {
    // A tile: 64 rows x 16 k  (thread -> row = tid/4, 4 consecutive k)
    {
      int row = threadIdx.x >> 2, kk = (threadIdx.x & 3) * 4;
      long r = r0 + row;
#pragma unroll
      for (int j = 0; j < 4; ++j) As[kk + j][row] = (r < R) ? to_f32(A[r * lda + k0 + kk + j]) : 0.f;
    }
    // W tile: 16 k x 64 n  (thread -> k = tid/16, 4 consecutive n)
    {
      int kk = threadIdx.x >> 4, nn = (threadIdx.x & 15) * 4;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        int n = n0 + nn + j;
        Bs[kk][nn + j] = (n < Nout) ? __ldg(W + (long)(k0 + kk) * ldw + n) : 0.f;
        if (DUAL) Bs2[kk][nn + j] = (n < Nout) ? __ldg(W2 + (long)(k0 + kk) * ldw + n) : 0.f;
      }
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < 16; ++kk) {
      float a[4], b[4], b2[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = As[kk][ty * 4 + i];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        b[j] = Bs[kk][tx * 4 + j];
        if (DUAL) b2[j] = Bs2[kk][tx * 4 + j];
      }
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
          if (DUAL) acc2[i][j] = fmaf(a[i], b2[j], acc2[i][j]);
        }
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    long r = r0 + ty * 4 + i;
    if (r >= R) continue;
    RowInfo ri = row_info(r, epi);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      int n = n0 + tx * 4 + j;
      if (n < Nout) epilogue_elem<T>(epi, ri, r, n, Nout, acc[i][j], acc2[i][j]);
    }
  }
}

template <typename T>
void launch_gemm_simt(const T* A, int lda, const float* W, const float* W2, int ldw, long R, int K, int Nout,
                      const Epi& epi, cudaStream_t st) {
  dim3 grid((unsigned)((R + 63) / 64), (unsigned)((Nout + 63) / 64));
  if (W2)
    gemm_simt_kernel<T, true><<<grid, 256, 0, st>>>(A, lda, W, W2, ldw, R, K, Nout, epi);
  else
    gemm_simt_kernel<T, false><<<grid, 256, 0, st>>>(A, lda, W, W2, ldw, R, K, Nout, epi);
}
template void launch_gemm_simt<float>(const float*, int, const float*, const float*, int, long, int, int, const Epi&, cudaStream_t);
template void launch_gemm_simt<bf16>(const bf16*, int, const float*, const float*, int, long, int, int, const Epi&, cudaStream_t);

// ---------------------------------------------------------------------------------------------
// Gated attention core (A.1/A.2/A.7/A.8 after the row permutation): one warp per query row.
//   qkg [(b,r,l), 3C] = [q/sqrt(d) | k | gate],  vt [((b,r),h,d), Lpad],  bias [(b,h,i), Lpad] or null,
//   keymask [b, L] in {0,1};  o[(b,r,i), h*32+d] = gate * sum_j softmax_j(q.k/sqrt(d) + bias + NEG) v
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(128) attn_simt_kernel(const T* __restrict__ qkg, const T* __restrict__ vt,
                                                        const T* __restrict__ bias, const float* __restrict__ keymask,
                                                        T* __restrict__ o, int B, int R, int L, int Lpad, int H) {
  extern __shared__ float sc[];   // [4 warps][L]
  int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int i = blockIdx.x * 4 + warp;
  int h = blockIdx.y;
  int br = blockIdx.z;           // b*R + r
  int b = br / R;
  if (i >= L) return;
  int C = H * 32;
  float* s = sc + warp * L;
  const T* qrow = qkg + ((long)br * L + i) * (3 * C) + h * 32;
  float q = to_f32(qrow[lane]);
  float mx = -INFINITY;
  for (int j = 0; j < L; ++j) {
    const T* krow = qkg + ((long)br * L + j) * (3 * C) + C + h * 32;
    float d = warp_sum(q * to_f32(krow[lane]));   // q already carries 1/sqrt(d) (R12)
    if (bias) d += to_f32(bias[(((long)b * H + h) * L + i) * Lpad + j]);
    d += 1e9f * (keymask[(long)b * L + j] - 1.0f);
    if (lane == 0) s[j] = d;
    mx = fmaxf(mx, d);
  }
  __syncwarp();
  float sum = 0.f;
  for (int j = lane; j < L; j += 32) {
    float e = expf(s[j] - mx);
    s[j] = e;
    sum += e;
  }
  sum = warp_sum(sum);
  __syncwarp();
  // lane = d
  const T* vrow = vt + (((long)br * H + h) * 32 + lane) * Lpad;
  float acc = 0.f;
  for (int j = 0; j < L; ++j) acc = fmaf(s[j], to_f32(vrow[j]), acc);
  float gate = to_f32(qrow[2 * C + lane]);
  store1(o + ((long)br * L + i) * C + h * 32 + lane, gate * acc / sum);
}

template <typename T>
void launch_attn_simt(const T* qkg, const T* vt, const T* bias, const float* keymask, T* o, int B, int R, int L,
                      int Lpad, int H, cudaStream_t st) {
  dim3 grid((L + 3) / 4, H, B * R);
  attn_simt_kernel<T><<<grid, 128, 4 * L * sizeof(float), st>>>(qkg, vt, bias, keymask, o, B, R, L, Lpad, H);
}
template void launch_attn_simt<float>(const float*, const float*, const float*, const float*, float*, int, int, int, int, int, cudaStream_t);
template void launch_attn_simt<bf16>(const bf16*, const bf16*, const bf16*, const float*, bf16*, int, int, int, int, int, cudaStream_t);

// ---------------------------------------------------------------------------------------------
// Triangle einsum (A.5 after the permutation): t[bc, i, j] = sum_k a[bc, i, k] b[bc, j, k]   (batched NT GEMM)
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) tri_einsum_simt_kernel(const T* __restrict__ a, const T* __restrict__ b,
                                                              float* __restrict__ t, int N, int Npad) {
  __shared__ float As[16][33], Bs[16][33];
  long base = (long)blockIdx.z * N * Npad;
  int i0 = blockIdx.y * 32, j0 = blockIdx.x * 32;
  int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;   // 16 x 16 threads, 2x2 each
  float acc[2][2] = {};
  for (int k0 = 0; k0 < N; k0 += 16) {
    for (int e = threadIdx.x; e < 512; e += 256) {
      int row = e >> 4, kk = e & 15;
      int k = k0 + kk;
      As[kk][row] = (i0 + row < N && k < N) ? to_f32(a[base + (long)(i0 + row) * Npad + k]) : 0.f;
      Bs[kk][row] = (j0 + row < N && k < N) ? to_f32(b[base + (long)(j0 + row) * Npad + k]) : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < 16; ++kk) {
      float a0 = As[kk][ty * 2], a1 = As[kk][ty * 2 + 1], b0 = Bs[kk][tx * 2], b1 = Bs[kk][tx * 2 + 1];
      acc[0][0] = fmaf(a0, b0, acc[0][0]);
      acc[0][1] = fmaf(a0, b1, acc[0][1]);
      acc[1][0] = fmaf(a1, b0, acc[1][0]);
      acc[1][1] = fmaf(a1, b1, acc[1][1]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int ii = 0; ii < 2; ++ii)
#pragma unroll
    for (int jj = 0; jj < 2; ++jj) {
      int i = i0 + ty * 2 + ii, j = j0 + tx * 2 + jj;
      if (i < N && j < N) t[base + (long)i * Npad + j] = acc[ii][jj];
    }
}

template <typename T>
void launch_tri_einsum_simt(const T* a_cm, const T* b_cm, float* t_cm, int batch, int N, int Npad, cudaStream_t st) {
  dim3 grid((N + 31) / 32, (N + 31) / 32, batch);
  tri_einsum_simt_kernel<T><<<grid, 256, 0, st>>>(a_cm, b_cm, t_cm, N, Npad);
}
template void launch_tri_einsum_simt<float>(const float*, const float*, float*, int, int, int, cudaStream_t);
template void launch_tri_einsum_simt<bf16>(const bf16*, const bf16*, float*, int, int, int, cudaStream_t);

// ---------------------------------------------------------------------------------------------
// LayerNorm across channels of the channel-major fp32 einsum output: t[(b,c), i, Npad] -> y[(b,i,j), C]
// Block = 32 positions (consecutive j) x C channels via shared memory.
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) lnc_kernel(const float* __restrict__ t, T* __restrict__ y,
                                                  const float* __restrict__ gamma, const float* __restrict__ beta,
                                                  const float* __restrict__ seq_mask, int C, int N, int Npad) {
  extern __shared__ float tile[];   // [C][33]
  int j0 = blockIdx.x * 32, i = blockIdx.y, b = blockIdx.z;
  if (seq_mask && seq_mask[(long)b * N + i] < 0.5f) return;   // padded row i: every output of it is at a masked position
  int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int c = warp; c < C; c += 8) {
    int j = j0 + lane;
    tile[c * 33 + lane] = (j < N) ? t[(((long)b * C + c) * N + i) * Npad + j] : 0.f;
  }
  __syncthreads();
  // warp w handles positions w, w+8, ... ; lanes over channels
  for (int p = warp; p < 32; p += 8) {
    int j = j0 + p;
    if (j >= N) continue;
    float s = 0.f;
    for (int c = lane; c < C; c += 32) s += tile[c * 33 + p];
    float mean = warp_sum(s) / C;
    float q = 0.f;
    for (int c = lane; c < C; c += 32) {
      float d = tile[c * 33 + p] - mean;
      q += d * d;
    }
    float rstd = rsqrtf(warp_sum(q) / C + 1e-5f);
    long row = ((long)b * N + i) * N + j;
    for (int c = lane; c < C; c += 32)
      store1(y + row * C + c, (tile[c * 33 + p] - mean) * rstd * __ldg(gamma + c) + __ldg(beta + c));
  }
}

// Streaming variant for C = 128 (the triangle hidden size): block = one (b, i) row x 64 consecutive j x 128 channels.
// Warp w loads channels [16 w, 16 w + 16) as 256-byte rows (float2 per lane: positions 2 lane, 2 lane + 1), so every thread
// holds 16 channels x 2 positions in registers; per-position statistics are the thread's partial sums combined across the
// eight warps through shared memory (no shuffles); the normalised values are staged [position][channel] in shared memory
// and leave as coalesced 16-byte stores.
__device__ __forceinline__ float2 lnc_ld2(const float* p) { return __ldg(reinterpret_cast<const float2*>(p)); }
__device__ __forceinline__ float2 lnc_ld2(const bf16* p) {
  const unsigned u = __ldg(reinterpret_cast<const unsigned*>(p));
  return __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&u));
}

template <typename T>
__global__ void __launch_bounds__(256) lnc128_kernel(const float* __restrict__ t, T* __restrict__ y,
                                                     const float* __restrict__ gamma, const float* __restrict__ beta,
                                                     const float* __restrict__ seq_mask, int N, int Npad) {
  constexpr int C = 128, PJ = 64;
  __shared__ float part[2][8][PJ];                       // [sum | sum of squares][warp][position]
  constexpr int ROWP = C + 16 / (int)sizeof(T);           // row pitch: + 16 bytes, so the packed 16-byte stores of the 32
                                                         // lanes (two rows apart) spread over the banks (2-way at worst)
  __shared__ __align__(16) T stage[PJ][ROWP];
  const int j0 = blockIdx.x * PJ, i = blockIdx.y, b = blockIdx.z;
  if (seq_mask && seq_mask[(long)b * N + i] < 0.5f) return;   // padded row i: every output of it is at a masked position
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int j = j0 + 2 * lane;
  float2 v[16];
  const bool in = j < Npad;                              // Npad is even: a pair never straddles the padded row end
#pragma unroll
  for (int k = 0; k < 16; ++k) {
    const int c = warp * 16 + k;
    v[k] = in ? lnc_ld2(t + (((long)b * C + c) * N + i) * Npad + j) : make_float2(0.f, 0.f);
  }
  float s0 = 0.f, s1 = 0.f;
#pragma unroll
  for (int k = 0; k < 16; ++k) {
    s0 += v[k].x;
    s1 += v[k].y;
  }
  part[0][warp][2 * lane] = s0;
  part[0][warp][2 * lane + 1] = s1;
  __syncthreads();
  float m0 = 0.f, m1 = 0.f;
#pragma unroll
  for (int w = 0; w < 8; ++w) {
    m0 += part[0][w][2 * lane];
    m1 += part[0][w][2 * lane + 1];
  }
  m0 *= (1.0f / C);
  m1 *= (1.0f / C);
  float q0 = 0.f, q1 = 0.f;
#pragma unroll
  for (int k = 0; k < 16; ++k) {
    const float d0 = v[k].x - m0, d1 = v[k].y - m1;
    q0 += d0 * d0;
    q1 += d1 * d1;
  }
  part[1][warp][2 * lane] = q0;
  part[1][warp][2 * lane + 1] = q1;
  __syncthreads();
  float r0 = 0.f, r1 = 0.f;
#pragma unroll
  for (int w = 0; w < 8; ++w) {
    r0 += part[1][w][2 * lane];
    r1 += part[1][w][2 * lane + 1];
  }
  r0 = rsqrtf(r0 * (1.0f / C) + 1e-5f);
  r1 = rsqrtf(r1 * (1.0f / C) + 1e-5f);
  {
    // this thread's 16 consecutive channels of its two positions: 16 * sizeof(T) contiguous bytes each, written as 16-byte packs
    __align__(16) T o0[16], o1[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const int c = warp * 16 + k;
      const float g = __ldg(gamma + c), be = __ldg(beta + c);
      store1(&o0[k], (v[k].x - m0) * r0 * g + be);
      store1(&o1[k], (v[k].y - m1) * r1 * g + be);
    }
    constexpr int NP = 16 * sizeof(T) / 16;              // 16-byte packs per position
#pragma unroll
    for (int q = 0; q < NP; ++q) {
      reinterpret_cast<uint4*>(&stage[2 * lane][warp * 16])[q] = reinterpret_cast<const uint4*>(o0)[q];
      reinterpret_cast<uint4*>(&stage[2 * lane + 1][warp * 16])[q] = reinterpret_cast<const uint4*>(o1)[q];
    }
  }
  __syncthreads();
  // PJ rows of C * sizeof(T) bytes, 16 bytes per thread and step
  constexpr int CH = C * sizeof(T) / 16;                 // 16-byte chunks per position
  for (int q = threadIdx.x; q < PJ * CH; q += 256) {
    const int pj = q / CH, ch = q % CH;
    if (j0 + pj < N)
      reinterpret_cast<uint4*>(y + (((long)b * N + i) * N + j0 + pj) * C)[ch] = reinterpret_cast<const uint4*>(&stage[pj][0])[ch];
  }
}

template <typename T>
void launch_lnc(const float* t_cm, T* y, const float* gamma, const float* beta, const float* seq_mask, int B, int C, int N,
                int Npad, cudaStream_t st) {
  if (C == 128) {
    dim3 grid((N + 63) / 64, N, B);
    lnc128_kernel<T><<<grid, 256, 0, st>>>(t_cm, y, gamma, beta, seq_mask, N, Npad);
    return;
  }
  dim3 grid((N + 31) / 32, N, B);
  lnc_kernel<T><<<grid, 256, C * 33 * sizeof(float), st>>>(t_cm, y, gamma, beta, seq_mask, C, N, Npad);
}
// The tcgen05 path's variant: bf16 channel-major einsum output -> fp16 rows (the next GEMM's A operand).  Block = one (b, i)
// row x 128 consecutive j x 128 channels; warp w owns channels [16 w, 16 w + 16), a lane four consecutive positions (one
// 8-byte load per channel: 256 bytes per warp load as in the fp32 variant), statistics across the eight warps through shared
// memory, normalised values staged [position][channel] and written as coalesced 16-byte stores.  (Measured alternatives: 16
// warps x 8 channels and values kept packed in registers were both slower.)
__global__ void __launch_bounds__(256) lnc128_bf16_kernel(const bf16* __restrict__ t, __half* __restrict__ y,
                                                          const float* __restrict__ gamma, const float* __restrict__ beta,
                                                          const float* __restrict__ seq_mask, int N, int Npad) {
  constexpr int C = 128, PJ = 128, ROWP = C + 8;
  __shared__ float part[2][8][PJ];
  __shared__ __align__(16) __half stage[PJ][ROWP];
  const int j0 = blockIdx.x * PJ, i = blockIdx.y, b = blockIdx.z;
  if (seq_mask && seq_mask[(long)b * N + i] < 0.5f) return;   // padded row i: every output of it is at a masked position
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int j = j0 + 4 * lane;
  const bool in = j < Npad;                              // Npad is a multiple of 8: a group of four never straddles the row end
  float v[16][4];
#pragma unroll
  for (int k = 0; k < 16; ++k) {
    const int c = warp * 16 + k;
    uint2 u = make_uint2(0u, 0u);
    if (in) u = __ldg(reinterpret_cast<const uint2*>(t + (((long)b * C + c) * N + i) * Npad + j));
    const float2 lo = __half22float2(*reinterpret_cast<const __half2*>(&u.x));   // the einsum output is fp16 (R17, round 2)
    const float2 hi = __half22float2(*reinterpret_cast<const __half2*>(&u.y));
    v[k][0] = lo.x; v[k][1] = lo.y; v[k][2] = hi.x; v[k][3] = hi.y;
  }
  float s[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
  for (int k = 0; k < 16; ++k)
#pragma unroll
    for (int p = 0; p < 4; ++p) s[p] += v[k][p];
  *reinterpret_cast<float4*>(&part[0][warp][4 * lane]) = make_float4(s[0], s[1], s[2], s[3]);
  __syncthreads();
  float m[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
  for (int w = 0; w < 8; ++w) {
    const float4 q = *reinterpret_cast<const float4*>(&part[0][w][4 * lane]);
    m[0] += q.x; m[1] += q.y; m[2] += q.z; m[3] += q.w;
  }
  float q2[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
  for (int p = 0; p < 4; ++p) m[p] *= (1.0f / C);
#pragma unroll
  for (int k = 0; k < 16; ++k)
#pragma unroll
    for (int p = 0; p < 4; ++p) {
      const float d = v[k][p] - m[p];
      q2[p] = fmaf(d, d, q2[p]);
    }
  *reinterpret_cast<float4*>(&part[1][warp][4 * lane]) = make_float4(q2[0], q2[1], q2[2], q2[3]);
  __syncthreads();
  float r[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
  for (int w = 0; w < 8; ++w) {
    const float4 q = *reinterpret_cast<const float4*>(&part[1][w][4 * lane]);
    r[0] += q.x; r[1] += q.y; r[2] += q.z; r[3] += q.w;
  }
#pragma unroll
  for (int p = 0; p < 4; ++p) r[p] = rsqrtf(r[p] * (1.0f / C) + 1e-5f);
  float g[16], be[16];
#pragma unroll
  for (int k = 0; k < 16; ++k) {
    g[k] = __ldg(gamma + warp * 16 + k);
    be[k] = __ldg(beta + warp * 16 + k);
  }
#pragma unroll
  for (int p = 0; p < 4; ++p) {
    __align__(16) __half o[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) o[k] = __float2half_rn((v[k][p] - m[p]) * r[p] * g[k] + be[k]);
    reinterpret_cast<uint4*>(&stage[4 * lane + p][warp * 16])[0] = reinterpret_cast<const uint4*>(o)[0];
    reinterpret_cast<uint4*>(&stage[4 * lane + p][warp * 16])[1] = reinterpret_cast<const uint4*>(o)[1];
  }
  __syncthreads();
  constexpr int CH = C * 2 / 16;                         // 16-byte chunks per position
  for (int q = threadIdx.x; q < PJ * CH; q += 256) {
    const int pj = q / CH, ch = q % CH;
    if (j0 + pj < N)
      reinterpret_cast<uint4*>(y + (((long)b * N + i) * N + j0 + pj) * C)[ch] = reinterpret_cast<const uint4*>(&stage[pj][0])[ch];
  }
}

// tcgen05 path: the einsum output is bf16 channel-major, C = 128, fp16 result (the next GEMM's A operand)
void launch_lnc_tc(const bf16* t_cm, __half* y, const float* gamma, const float* beta, const float* seq_mask, int B, int N,
                   int Npad, cudaStream_t st) {
  dim3 grid((N + 127) / 128, N, B);
  lnc128_bf16_kernel<<<grid, 256, 0, st>>>(t_cm, y, gamma, beta, seq_mask, N, Npad);
}
template void launch_lnc<float>(const float*, float*, const float*, const float*, const float*, int, int, int, int, cudaStream_t);
template void launch_lnc<bf16>(const float*, bf16*, const float*, const float*, const float*, int, int, int, int, cudaStream_t);
template void launch_lnc<__half>(const float*, __half*, const float*, const float*, const float*, int, int, int, int, cudaStream_t);

// ---------------------------------------------------------------------------------------------
// Outer-product-mean core (A.4): one block per (b, i, j).  a, b: [(b,s,i), c_opm] already masked by mu.
//   z[b,i,j,:] += ( vec(sum_s a[s,i] (x) b[s,j]) / (1e-3 + n_ij) ) Wout + bout,   n_ij = sum_s mu_si mu_sj
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) opm_simt_kernel(const T* __restrict__ a, const T* __restrict__ bb,
                                                       const float* __restrict__ wout, const float* __restrict__ bout,
                                                       const float* __restrict__ seq_mask,
                                                       const float* __restrict__ msa_mask, float* __restrict__ z, int S,
                                                       int N, int co, int cz) {
  extern __shared__ float O[];   // [co*co]
  int j = blockIdx.x, i = blockIdx.y, b = blockIdx.z;
  for (int e = threadIdx.x; e < co * co; e += blockDim.x) {
    int c1 = e / co, c2 = e % co;
    float acc = 0.f;
    for (int s = 0; s < S; ++s)
      acc = fmaf(to_f32(a[(((long)b * S + s) * N + i) * co + c1]), to_f32(bb[(((long)b * S + s) * N + j) * co + c2]), acc);
    O[e] = acc;
  }
  float n = 0.f;
  for (int s = 0; s < S; ++s) n += msa_mask[(long)b * S + s];
  n *= seq_mask[(long)b * N + i] * seq_mask[(long)b * N + j];
  float inv = 1.0f / (1e-3f + n);
  __syncthreads();
  for (int e = threadIdx.x; e < cz; e += blockDim.x) {
    float acc = 0.f;
    for (int k = 0; k < co * co; ++k) acc = fmaf(O[k], __ldg(wout + (long)k * cz + e), acc);
    long idx = (((long)b * N + i) * N + j) * cz + e;
    z[idx] += acc * inv + __ldg(bout + e);
  }
}

template <typename T>
void launch_opm_simt(const T* a, const T* b, const float* wout, const float* bout, const float* seq_mask,
                     const float* msa_mask, float* z, int B, int S, int N, int c_opm, int c_z, cudaStream_t st) {
  dim3 grid(N, N, B);
  opm_simt_kernel<T><<<grid, 256, c_opm * c_opm * sizeof(float), st>>>(a, b, wout, bout, seq_mask, msa_mask, z, S, N,
                                                                       c_opm, c_z);
}
template void launch_opm_simt<float>(const float*, const float*, const float*, const float*, const float*, const float*, float*, int, int, int, int, int, cudaStream_t);
template void launch_opm_simt<bf16>(const bf16*, const bf16*, const float*, const float*, const float*, const float*, float*, int, int, int, int, int, cudaStream_t);


// ---------------------------------------------------------------------------------------------
// Pair-bias heads of the MSA row attention (A.1):  bias[b, h, i, j] = scale * sum_c LN'(z[b,i,j])_c W[c, h],  c_z = 128, H <= 8.
// 512 bytes in and 2 H bytes out per pair with 2 H c_z FLOP: HBM-bound streaming work (as a launch of the projection GEMM it
// ran at 2.3 TB/s, paced by that kernel's LayerNorm producers; a first SIMT version with the eight dot products on the FMA
// pipes was bound by instruction issue: 107 warp instructions per row, 2.7 TB/s).  This version: a warp owns 16 consecutive
// pair rows and holds them in the A-fragment layout of mma.sync.m16n8k16 (lane = (row group g, column group t): rows g and
// g + 8, columns 16 kb + 2 t + {0, 1, 8, 9} of every 16-wide k-block, loaded as float2), normalises in registers (statistics
// over the four lanes of a row: two shuffles each), converts xhat to fp16 pairs and issues eight mma.sync against the weight
// fragments, which hold gamma_c W[c, h] scale as fp16 (LN'(z) W = xhat (gamma . W) + beta W: the affine part of the
// LayerNorm moves into the weights, the constant beta W is added in fp32 at the end; fp16 operands as the projection GEMM,
// R17).  Pairs with a masked i or j are skipped: the attention masks key j itself and a masked query's output is
// unspecified (R3); what the bias buffer holds there is a finite older value.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void mma_16816_f16(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t pack_h2(float a, float b) {
  __half2 h = __floats2half2_rn(a, b);
  return *reinterpret_cast<uint32_t*>(&h);
}
__device__ __forceinline__ float2 ld_nc_f2(const float2* p) {
  float2 r;
  asm volatile("ld.global.nc.L1::no_allocate.v2.f32 {%0,%1}, [%2];" : "=f"(r.x), "=f"(r.y) : "l"(p));
  return r;
}

constexpr int LH_WARPS = 8;   // 16 pair rows per warp and iteration
__global__ void __launch_bounds__(32 * LH_WARPS, 2) ln_heads128_kernel(const float* __restrict__ z, const float* __restrict__ gamma,
                                                                       const float* __restrict__ beta, const float* __restrict__ W,
                                                                       float scale, const float* __restrict__ seq_mask,
                                                                       bf16* __restrict__ out, int B, int N, int Lpad, int H) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, g = lane >> 2, t = lane & 3;
  // B fragments of the eight k-blocks: b0 = (k = 16 kb + 2t, +1; n = g), b1 = (k = 16 kb + 2t + 8, +9; n = g), n = head
  uint32_t bw[8][2];
  float bias_h[2] = {0.f, 0.f};                 // beta W scale for this lane's two output heads (2t, 2t + 1)
#pragma unroll
  for (int kb = 0; kb < 8; ++kb) {
#pragma unroll
    for (int hf = 0; hf < 2; ++hf) {
      const int c = 16 * kb + 2 * t + 8 * hf;
      const float w0 = g < H ? __ldg(gamma + c) * __ldg(W + c * H + g) * scale : 0.f;
      const float w1 = g < H ? __ldg(gamma + c + 1) * __ldg(W + (c + 1) * H + g) * scale : 0.f;
      bw[kb][hf] = pack_h2(w0, w1);
    }
  }
  {
    float part[8];
#pragma unroll
    for (int hh = 0; hh < 8; ++hh) {
      part[hh] = 0.f;
      if (hh < H)
        for (int c = lane * 4; c < lane * 4 + 4; ++c) part[hh] = fmaf(__ldg(beta + c) * scale, __ldg(W + c * H + hh), part[hh]);
      part[hh] = warp_sum(part[hh]);
    }
#pragma unroll
    for (int hh = 0; hh < 8; ++hh) {
      if (hh == 2 * t) bias_h[0] = part[hh];
      if (hh == 2 * t + 1) bias_h[1] = part[hh];
    }
  }
  const long rows = (long)B * N * N;
  for (long r0 = ((long)blockIdx.x * LH_WARPS + warp) * 16; r0 < rows; r0 += (long)gridDim.x * LH_WARPS * 16) {
    bool on[2];
    long oidx[2];   // output index of head 0 (rows < 2^32 is checked by the launcher: 32-bit divisions only)
    const float* src[2];
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      const long r = r0 + g + 8 * q;
      on[q] = false;
      oidx[q] = 0;
      src[q] = z;
      if (r < rows) {
        const unsigned ru = (unsigned)r, bx = ru / (unsigned)N, y = ru - bx * (unsigned)N, b = bx / (unsigned)N, x = bx - b * (unsigned)N;
        on[q] = seq_mask[bx] > 0.5f && seq_mask[b * (unsigned)N + y] > 0.5f;
        oidx[q] = ((long)b * H * N + x) * (long)Lpad + y;
        src[q] = z + r * 128;
      }
    }
    if (!__any_sync(0xffffffffu, on[0] || on[1])) continue;
    float2 v[2][8][2];
#pragma unroll
    for (int q = 0; q < 2; ++q)
#pragma unroll
      for (int kb = 0; kb < 8; ++kb)
#pragma unroll
        for (int hf = 0; hf < 2; ++hf)
          v[q][kb][hf] = on[q] ? ld_nc_f2(reinterpret_cast<const float2*>(src[q] + 16 * kb + 2 * t + 8 * hf)) : make_float2(0.f, 0.f);
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    float rstd[2], nm[2];
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      float s = 0.f;
#pragma unroll
      for (int kb = 0; kb < 8; ++kb) s += (v[q][kb][0].x + v[q][kb][0].y) + (v[q][kb][1].x + v[q][kb][1].y);
      s += __shfl_xor_sync(0xffffffffu, s, 1);
      s += __shfl_xor_sync(0xffffffffu, s, 2);
      const float mean = s * (1.0f / 128);
      float qq = 0.f;
#pragma unroll
      for (int kb = 0; kb < 8; ++kb) {
        const float a = v[q][kb][0].x - mean, b = v[q][kb][0].y - mean, c = v[q][kb][1].x - mean, d = v[q][kb][1].y - mean;
        qq += (a * a + b * b) + (c * c + d * d);
      }
      qq += __shfl_xor_sync(0xffffffffu, qq, 1);
      qq += __shfl_xor_sync(0xffffffffu, qq, 2);
      rstd[q] = rsqrtf(qq * (1.0f / 128) + 1e-5f);
      nm[q] = -mean * rstd[q];
    }
#pragma unroll
    for (int kb = 0; kb < 8; ++kb) {
      uint32_t a[4];   // a0 (row g, cols 2t..), a1 (row g + 8, cols 2t..), a2 (row g, cols 2t + 8..), a3 (row g + 8, cols 2t + 8..)
      a[0] = pack_h2(fmaf(v[0][kb][0].x, rstd[0], nm[0]), fmaf(v[0][kb][0].y, rstd[0], nm[0]));
      a[1] = pack_h2(fmaf(v[1][kb][0].x, rstd[1], nm[1]), fmaf(v[1][kb][0].y, rstd[1], nm[1]));
      a[2] = pack_h2(fmaf(v[0][kb][1].x, rstd[0], nm[0]), fmaf(v[0][kb][1].y, rstd[0], nm[0]));
      a[3] = pack_h2(fmaf(v[1][kb][1].x, rstd[1], nm[1]), fmaf(v[1][kb][1].y, rstd[1], nm[1]));
      mma_16816_f16(acc, a, bw[kb][0], bw[kb][1]);
    }
    // acc: (row g, head 2t), (row g, head 2t + 1), (row g + 8, head 2t), (row g + 8, head 2t + 1)
    const long hs = (long)N * Lpad;
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      if (on[q]) {
        __half* oh = reinterpret_cast<__half*>(out);   // the pair bias is held as fp16 (R17): 8x finer than bf16 at |bias| ~ 1
        if (2 * t < H) oh[oidx[q] + (long)(2 * t) * hs] = __float2half_rn(acc[2 * q] + bias_h[0]);
        if (2 * t + 1 < H) oh[oidx[q] + (long)(2 * t + 1) * hs] = __float2half_rn(acc[2 * q + 1] + bias_h[1]);
      }
    }
  }
}

void launch_ln_heads128(const float* z, const float* gamma, const float* beta, const float* W, float scale, const float* seq_mask,
                        bf16* out, int B, int N, int Lpad, int H, int num_sms, cudaStream_t st) {
  const long rows = (long)B * N * N, blocks = (rows + LH_WARPS * 16 - 1) / (LH_WARPS * 16);
  const long cap = (long)num_sms * 2;   // persistent: two CTAs per SM, the weight fragments are built once per CTA
  ln_heads128_kernel<<<(unsigned)(blocks < cap ? blocks : cap), 32 * LH_WARPS, 0, st>>>(z, gamma, beta, W, scale, seq_mask, out, B, N,
                                                                                        Lpad, H);
}

// ---------------------------------------------------------------------------------------------
// Outer-product-mean operands (A.4):  ab_t[(b, i), ch, s] = mu_si (LN(m_si) [W_a | W_b] + [b_a | b_b])_ch,  c_m = 256, 64 columns,
// written transposed (s contiguous) for the outer-product kernel.  1 KB in and 128 bytes out per (s, i) with 32 K FLOP: HBM-bound
// (as a launch of the projection GEMM it ran at 2.6-2.7 TB/s, paced by that kernel's LayerNorm producers).  Same scheme as the
// pair-bias heads above: a warp owns 16 consecutive sequences s of one residue (b, i) and keeps the 16 x 256 fp32 values in
// registers in the A-fragment layout of mma.sync.m16n8k16 (128 registers per lane), normalises them there, and multiplies by
// gamma . W held as fp16 B fragments in shared memory (32 KB, laid out per lane so that a fragment fetch is four conflict-free
// 16-byte loads); beta W + bias is added in fp32.  Residues i that are padded are skipped; masked sequences of an unmasked
// residue are written as exact zeros (they are summed over without a softmax).
// ---------------------------------------------------------------------------------------------
constexpr int OA_WARPS = 8;
__global__ void __launch_bounds__(32 * OA_WARPS, 1)
ln_opm_ab256_kernel(const float* __restrict__ msa, const float* __restrict__ gamma, const float* __restrict__ beta,
                    const float* __restrict__ Wa, const float* __restrict__ Wb, const float* __restrict__ ba,
                    const float* __restrict__ bb, const float* __restrict__ seq_mask, const float* __restrict__ msa_mask,
                    bf16* __restrict__ out, int B, int S, int N, int Spad) {
  __shared__ uint4 wfrag[16 * 4 * 32];      // [kb][q][lane]: 16 bytes = fragments (nt = 2q, 2q + 1) x (b0, b1) of this lane
  __shared__ float cst[64];                 // beta W + bias
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, g = lane >> 2, t = lane & 3;
  auto wcol = [&](int c, int n) { return n < 32 ? __ldg(Wa + c * 32 + n) : __ldg(Wb + c * 32 + n - 32); };
  for (int e = threadIdx.x; e < 16 * 4 * 32; e += blockDim.x) {
    const int ln = e & 31, q = (e >> 5) & 3, kb = e >> 7, gg = ln >> 2, tt = ln & 3;
    uint32_t w[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {           // j = (nt - 2q) * 2 + hf
      const int n = 8 * (2 * q + (j >> 1)) + gg, c = 16 * kb + 2 * tt + 8 * (j & 1);
      w[j] = pack_h2(__ldg(gamma + c) * wcol(c, n), __ldg(gamma + c + 1) * wcol(c + 1, n));
    }
    wfrag[e] = make_uint4(w[0], w[1], w[2], w[3]);
  }
  if (threadIdx.x < 64) {
    const int n = threadIdx.x;
    float a = n < 32 ? __ldg(ba + n) : __ldg(bb + n - 32);
    for (int c = 0; c < 256; ++c) a = fmaf(__ldg(beta + c), wcol(c, n), a);
    cst[n] = a;
  }
  __syncthreads();
  const int sblocks = (S + 15) / 16;
  const long units = (long)B * N * sblocks;
  for (long u = (long)blockIdx.x * OA_WARPS + warp; u < units; u += (long)gridDim.x * OA_WARPS) {
    const int sb = (int)(u % sblocks);
    const long bi = u / sblocks;            // b * N + i
    if (!(seq_mask[bi] > 0.5f)) continue;   // padded residue: nothing of this unit is read later
    const int b = (int)(bi / N), i = (int)(bi - (long)b * N);
    bool on[2], inr[2];
    const float* src[2];
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      const int sq = sb * 16 + g + 8 * q;
      inr[q] = sq < S;
      on[q] = inr[q] && msa_mask[(long)b * S + sq] > 0.5f;
      src[q] = msa + (((long)b * S + (inr[q] ? sq : 0)) * N + i) * 256;
    }
    float2 v[2][16][2];
#pragma unroll
    for (int q = 0; q < 2; ++q)
#pragma unroll
      for (int kb = 0; kb < 16; ++kb)
#pragma unroll
        for (int hf = 0; hf < 2; ++hf)
          v[q][kb][hf] = on[q] ? ld_nc_f2(reinterpret_cast<const float2*>(src[q] + 16 * kb + 2 * t + 8 * hf)) : make_float2(0.f, 0.f);
    float rstd[2], nm[2];
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      float sm = 0.f;
#pragma unroll
      for (int kb = 0; kb < 16; ++kb) sm += (v[q][kb][0].x + v[q][kb][0].y) + (v[q][kb][1].x + v[q][kb][1].y);
      sm += __shfl_xor_sync(0xffffffffu, sm, 1);
      sm += __shfl_xor_sync(0xffffffffu, sm, 2);
      const float mean = sm * (1.0f / 256);
      float qq = 0.f;
#pragma unroll
      for (int kb = 0; kb < 16; ++kb) {
        const float a = v[q][kb][0].x - mean, bq = v[q][kb][0].y - mean, c = v[q][kb][1].x - mean, d = v[q][kb][1].y - mean;
        qq += (a * a + bq * bq) + (c * c + d * d);
      }
      qq += __shfl_xor_sync(0xffffffffu, qq, 1);
      qq += __shfl_xor_sync(0xffffffffu, qq, 2);
      rstd[q] = rsqrtf(qq * (1.0f / 256) + 1e-5f);
      nm[q] = -mean * rstd[q];
    }
    float acc[8][4];
#pragma unroll
    for (int nt = 0; nt < 8; ++nt)
#pragma unroll
      for (int e = 0; e < 4; ++e) acc[nt][e] = 0.f;
#pragma unroll
    for (int kb = 0; kb < 16; ++kb) {
      uint32_t a[4];
      a[0] = pack_h2(fmaf(v[0][kb][0].x, rstd[0], nm[0]), fmaf(v[0][kb][0].y, rstd[0], nm[0]));
      a[1] = pack_h2(fmaf(v[1][kb][0].x, rstd[1], nm[1]), fmaf(v[1][kb][0].y, rstd[1], nm[1]));
      a[2] = pack_h2(fmaf(v[0][kb][1].x, rstd[0], nm[0]), fmaf(v[0][kb][1].y, rstd[0], nm[0]));
      a[3] = pack_h2(fmaf(v[1][kb][1].x, rstd[1], nm[1]), fmaf(v[1][kb][1].y, rstd[1], nm[1]));
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const uint4 w = wfrag[(kb * 4 + q) * 32 + lane];
        mma_16816_f16(acc[2 * q], a, w.x, w.y);
        mma_16816_f16(acc[2 * q + 1], a, w.z, w.w);
      }
    }
    // acc[nt]: (row g, col 8 nt + 2t), (g, + 1), (row g + 8, col 8 nt + 2t), (g + 8, + 1); rows = sequences, written transposed
    __half* ohalf = reinterpret_cast<__half*>(out) + (bi * 64) * (long)Spad;   // fp16 operands (R17 round 2)
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      if (!inr[q]) continue;
      const int sq = sb * 16 + g + 8 * q;
#pragma unroll
      for (int nt = 0; nt < 8; ++nt) {
        const int col = 8 * nt + 2 * t;
        ohalf[(long)col * Spad + sq] = __float2half_rn(on[q] ? acc[nt][2 * q] + cst[col] : 0.f);
        ohalf[(long)(col + 1) * Spad + sq] = __float2half_rn(on[q] ? acc[nt][2 * q + 1] + cst[col + 1] : 0.f);
      }
    }
  }
}

void launch_ln_opm_ab256(const float* msa, const float* gamma, const float* beta, const float* Wa, const float* Wb, const float* ba,
                         const float* bb, const float* seq_mask, const float* msa_mask, bf16* out, int B, int S, int N, int Spad,
                         int num_sms, cudaStream_t st) {
  const long units = (long)B * N * ((S + 15) / 16), blocks = (units + OA_WARPS - 1) / OA_WARPS;
  ln_opm_ab256_kernel<<<(unsigned)(blocks < num_sms ? blocks : num_sms), 32 * OA_WARPS, 0, st>>>(msa, gamma, beta, Wa, Wb, ba, bb, seq_mask,
                                                                                                msa_mask, out, B, S, N, Spad);
}

}  // namespace pf
