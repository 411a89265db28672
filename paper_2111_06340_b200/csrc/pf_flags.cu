// Mask-derived work flags (PF_BF16 path).  Proteins are padded to their bucket (one compiled model serves
// proteins of similar length); a 128-row tile of a projection, or an attention unit, all of whose rows are masked
// (padded residues, masked MSA rows) produces only outputs at masked positions, which are unspecified (R3) and enter
// every later sum with an exactly-zero weight.  Such tiles / units are skipped; what they would have written stays at
// the (finite: the workspace is zero-filled at allocation) value it had.  Key tiles past the last unmasked key are
// skipped as well (exact: their softmax weights are exactly 0).  Exception: operands that are contracted over a masked
// index without a softmax (triangle einsum over k, outer product over s) must be exactly zero there, so their projection
// tiles are skipped only when the KEPT index is padded (kind 3).
#include "pf_internal.h"

namespace pf {

// kind: 0 rows (b, s=x, i=y) of the MSA: rho_x sigma_y | 1 rows (b, i=x, s=y): sigma_x rho_y | 2 pair rows: sigma_x sigma_y
//       3 rows (b, i=x, y) whose y index is CONTRACTED later (k of the triangle einsum, s of the outer product): only a
//         padded residue x makes the row skippable; entries at masked y must be written (as exact zeros)
__device__ __forceinline__ bool row_active(const float* seq_mask, const float* msa_mask, int kind, int b, int x, int y, int D1,
                                           int D2) {
  if (kind == 3) return seq_mask[(long)b * D1 + x] > 0.5f;
  const float mx = (kind == 0 ? msa_mask : seq_mask)[(long)b * D1 + x];
  const float my = (kind == 1 ? msa_mask : seq_mask)[(long)b * D2 + y];
  return mx * my > 0.5f;
}

// One thread per tile.  YT > 0: tile = XT consecutive x times YT consecutive y of one b (gemm2 geometry);
// YT == 0: tile = 128 consecutive rows of the [B*D1*D2] row list (transition kernel).
__global__ void tile_flags_kernel(const float* __restrict__ seq_mask, const float* __restrict__ msa_mask, int kind, int B,
                                  int D1, int D2, int XT, int YT, unsigned char* __restrict__ flags, long num_tiles) {
  const long t = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= num_tiles) return;
  bool any = false;
  if (YT > 0) {
    const int tiles_y = (D2 + YT - 1) / YT, tiles_x = (D1 + XT - 1) / XT;
    const int ty = (int)(t % tiles_y);
    const long tx = t / tiles_y;
    const int b = (int)(tx / tiles_x);
    const int x0 = (int)(tx - (long)b * tiles_x) * XT, y0 = ty * YT;
    for (int x = x0; x < x0 + XT && x < D1 && !any; ++x)
      for (int y = y0; y < y0 + YT && y < D2; ++y)
        if (row_active(seq_mask, msa_mask, kind, b, x, y, D1, D2)) {
          any = true;
          break;
        }
  } else {
    const long R = (long)B * D1 * D2, per = (long)D1 * D2;
    for (long r = t * 128; r < t * 128 + 128 && r < R; ++r) {
      const int b = (int)(r / per);
      const int rem = (int)(r - (long)b * per);
      if (row_active(seq_mask, msa_mask, kind, b, rem / D2, rem % D2, D1, D2)) {
        any = true;
        break;
      }
    }
  }
  flags[t] = any ? 1 : 0;
}

// key_tiles[b] = number of 64-key tiles up to and including the last unmasked key of mask[b, 0..L) (at least 1)
__global__ void key_tiles_kernel(const float* __restrict__ mask, int B, int L, int* __restrict__ key_tiles) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= B) return;
  int last = 0;
  for (int j = 0; j < L; ++j)
    if (mask[(long)b * L + j] > 0.5f) last = j;
  key_tiles[b] = last / 64 + 1;
}

// Order-preserving compaction of the rows (b, r) of an attention launch that have at least one unmasked query:
// rows[k] = {b*R + r, key tiles to visit for protein b}, *n_rows = their number.  One block; B*R <= 65535.
__global__ void __launch_bounds__(1024) row_list_kernel(const float* __restrict__ rowmask, const int* __restrict__ key_tiles,
                                                        int B, int R, int2* __restrict__ rows, int* __restrict__ n_rows) {
  __shared__ int warp_sums[32];
  __shared__ int total;
  const int n = B * R, per = (n + 1023) / 1024;
  const int lo = threadIdx.x * per, hi = min(lo + per, n);
  int cnt = 0;
  for (int i = lo; i < hi; ++i) cnt += rowmask[i] > 0.5f ? 1 : 0;
  // block exclusive scan of cnt
  int incl = cnt;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int t = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += t;
  }
  if (lane == 31) warp_sums[warp] = incl;
  __syncthreads();
  if (warp == 0) {
    int w = warp_sums[lane], wi = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int t = __shfl_up_sync(0xffffffffu, wi, o);
      if (lane >= o) wi += t;
    }
    warp_sums[lane] = wi - w;
    if (lane == 31) total = wi;
  }
  __syncthreads();
  int pos = warp_sums[warp] + incl - cnt;
  for (int i = lo; i < hi; ++i)
    if (rowmask[i] > 0.5f) rows[pos++] = make_int2(i, key_tiles[i / R]);
  if (threadIdx.x == 0) *n_rows = total;
}

void launch_row_list(const float* rowmask, const int* key_tiles, int B, int R, void* rows, int* n_rows, cudaStream_t st) {
  row_list_kernel<<<1, 1024, 0, st>>>(rowmask, key_tiles, B, R, reinterpret_cast<int2*>(rows), n_rows);
}

void launch_tile_flags(const float* seq_mask, const float* msa_mask, int kind, int B, int D1, int D2, int XT, int YT,
                       unsigned char* flags, long num_tiles, cudaStream_t st) {
  const int threads = 128;
  tile_flags_kernel<<<(unsigned)((num_tiles + threads - 1) / threads), threads, 0, st>>>(seq_mask, msa_mask, kind, B, D1, D2,
                                                                                        XT, YT, flags, num_tiles);
}
void launch_key_tiles(const float* mask, int B, int L, int* key_tiles, cudaStream_t st) {
  key_tiles_kernel<<<(B + 127) / 128, 128, 0, st>>>(mask, B, L, key_tiles);
}

}  // namespace pf
