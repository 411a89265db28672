// Gated attention core on tcgen05 tensor cores (sm_100a), shared by MSA row attention with pair bias (A.1), MSA
// column attention (A.2) and triangle attention around the starting / ending node (A.7 / A.8) after the driver's row
// permutation:  for every (b, r, h) and query i
//     o[i, :] = gate[i, :] * sum_j softmax_j( q[i].k[j] + bias[b, h, i, j] + NEG(keymask[b, j]) ) v[j, :]
// (q already carries log2(e)/sqrt(d) and the bias log2(e), R12: the softmax runs in the exp2 domain).  Flash-style: logits
// never leave the SM (north_star: "no materialised N^3 logits").  Persistent CTAs, two per SM; a work unit is one
// (b*r, h, 128-query tile), its key tiles of 64 are the pipeline steps, and steps run back to back across units:
//   warp 4 (TMA)   Q (double buffered per unit) and per step {K 64x32 (64B swizzle), V^T 32x64, bias 128x64 (128B swizzle)}
//                  through a ring, running ahead of the consumers by the ring depth
//   warp 5 (MMA)   S(i+1) = Q K^T + bias I  (M=128 N=64; K=2x16 for Q K^T, then the bf16 pair-bias tile [128 x 64] times a
//                  constant 64 x 64 identity, K=4x16: the tensor core adds the bias exactly (fp32 accumulation), so the softmax
//                  warps never unpack it; TMEM double buffered) is issued BEFORE waiting for P(i), so the
//                  tensor core works on the next logits while the softmax warps are busy; O_tile = P V (M=128 N=32 K=4x16)
//   warps 0-3      thread-per-row online softmax in fp32 from tcgen05.ld (ex2.approx), P (bf16 pairs) written back over the
//                  logits in tensor memory (tcgen05.st) and read by P V as a TMEM A operand.  O accumulates in TMEM over the key tiles of a unit (P V with accumulate); P is taken
//                  relative to a reference maximum that moves only when the running maximum has grown by more than 2^8, and
//                  only then is O rescaled (tcgen05.ld, multiply, tcgen05.st) — the time of this kernel follows the
//                  instruction count of these warps, and the per-tile "(O + PV) alpha" round trip through registers was 15 %
//                  of it; gate (prefetched at unit start) and 1/l applied at the end, 64-byte row stores.
// ~96 KB of shared memory and 256 TMEM columns per CTA -> 2 CTAs per SM overlap each other's softmax and barrier latency.
#include "pf_internal.h"
#include "pf_device.cuh"
#include "pf_tc.cuh"

namespace pf {

int tma_encode_bf16(TmaCtx* ctx, CUtensorMap* out, const void* base, int rank, const uint64_t* dims,
                    const uint64_t* strides_elems, const uint32_t* box, int swizzle_bytes);

constexpr int AT_BQ = 128;        // queries per unit
constexpr int AT_BK = 64;         // keys per step
constexpr int AT_THREADS = 192;   // 4 softmax warps + TMA warp + MMA warp
constexpr int AT_MAXKEYS = 1024;  // mask terms kept in shared memory

struct AttnSmem {
  static constexpr int Q_BYTES = AT_BQ * 64;                       // 128 x 32 bf16, 64B swizzle: 8 KB
  static constexpr int Q_OFF = 0;                                  // two Q buffers
  static constexpr int STAGE_OFF = Q_OFF + 2 * Q_BYTES;
  static constexpr int K_BYTES = AT_BK * 64;                       // 64 x 32 bf16: 4 KB
  static constexpr int V_BYTES = 32 * 128;                         // 32 x 64 bf16: 4 KB
  static constexpr int B_BYTES = AT_BQ * 128;                      // 128 x 64 bf16: 16 KB
  static constexpr int POOL_BYTES = 72 * 1024;                     // 3 stages with a bias tile, 8 without (one is unused)
  static constexpr int MAX_STAGES = 8;
  static constexpr int ID_OFF = STAGE_OFF + POOL_BYTES;            // 64 x 64 bf16 identity, K-major 128B swizzle: 8 KB
  static constexpr int MASK_OFF = ID_OFF + 64 * 128;               // one bit per key: 1 = masked or out of range
  static constexpr int BAR_OFF = MASK_OFF + AT_MAXKEYS / 8;
  // No alignment slack: two CTAs per SM must fit (98,688 B each).  The dynamic shared memory window of a kernel
  // without static shared memory starts 1024-byte aligned; the kernel traps if it ever does not.
  static constexpr int TOTAL = BAR_OFF + 256;
};

struct AttnParams {
  const bf16* qkg;
  const float* keymask;
  bf16* o;
  int R, L, H, QT, n_kt, has_bias, stages, stage_bytes;
  const int2* rows;        // device list {b*R + r, key tiles to visit} of the rows with an unmasked query (pf_flags.cu)
  const int* n_rows;       // device scalar: its length
};

// Work unit u -> (row entry, head, query tile); the row entry is a plain load (no data-dependent branch), so every role
// fetches the NEXT unit's entry at the top of the current unit and the load latency is off its critical path.
__device__ __forceinline__ int2 attn_row_entry(int u, int units, const AttnParams& p) {
  return u < units ? __ldg(p.rows + u / (p.QT * p.H)) : make_int2(0, 0);
}

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

__global__ void __launch_bounds__(AT_THREADS, 2)
attn_tc_kernel(const __grid_constant__ CUtensorMap tmQK, const __grid_constant__ CUtensorMap tmV,
               const __grid_constant__ CUtensorMap tmBias, const __grid_constant__ AttnParams p) {
  using SM = AttnSmem;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = smem_raw;
  if (tc::smem_u32(smem_raw) & 1023u) __trap();
  uint32_t* mbits = reinterpret_cast<uint32_t*>(smem + SM::MASK_OFF);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + SM::BAR_OFF);
  uint64_t* q_full = bars;                       // [2]
  uint64_t* q_empty = bars + 2;                  // [2]
  uint64_t* kv_full = bars + 4;                  // [MAX_STAGES]
  uint64_t* kv_empty = kv_full + SM::MAX_STAGES; // [MAX_STAGES]
  uint64_t* s_full = kv_empty + SM::MAX_STAGES;  // [2]
  uint64_t* p_full = s_full + 2;
  uint64_t* o_full = p_full + 1;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(o_full + 1);
  uint32_t* maskbits = tmem_slot + 1;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int C = p.H * 32;
  const int ST = p.stages;

  if (warp == 4 && lane == 0) {
    tc::prefetch_tmap(&tmQK);
    tc::prefetch_tmap(&tmV);
    if (p.has_bias) tc::prefetch_tmap(&tmBias);
    for (int i = 0; i < 2; ++i) {
      tc::mbar_init(&q_full[i], 1);
      tc::mbar_init(&q_empty[i], 1);
      tc::mbar_init(&s_full[i], 1);
    }
    for (int s = 0; s < SM::MAX_STAGES; ++s) {
      tc::mbar_init(&kv_full[s], 1);
      tc::mbar_init(&kv_empty[s], 1);
    }
    tc::mbar_init(p_full, 128);
    tc::mbar_init(o_full, 1);
    tc::fence_barrier_init();
  }
  if (warp == 5) tc::tmem_alloc<256>(tmem_slot);
  if (p.has_bias) {
    // identity operand of the bias MMA: element (j, k) of a K-major [64 x 64] bf16 tile, 1.0 on the diagonal
    uint32_t* idw = reinterpret_cast<uint32_t*>(smem + SM::ID_OFF);
    for (int i = threadIdx.x; i < 64 * 128 / 4; i += AT_THREADS) idw[i] = 0u;
    __syncthreads();
    if (threadIdx.x < 64) {
      const int j = threadIdx.x;
      *reinterpret_cast<uint16_t*>(smem + SM::ID_OFF + tc::swz_offset<128>(j, j >> 3) + (j & 7) * 2) = 0x3C00;   // fp16 1.0: the pair bias is stored as fp16 (R17)
    }
    tc::fence_proxy_async_smem();
  }
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const uint32_t tmem_S = tmem_base, tmem_O = tmem_base + 128;   // S[2] at columns 0 / 64, O at [128, 160)

  if (warp == 4) {
    // ============================================================= TMA producer
    if (tc::elect_one()) {
      const uint32_t stage_tx = SM::K_BYTES + SM::V_BYTES + (p.has_bias ? SM::B_BYTES : 0);
      uint32_t uc = 0, s = 0, sph = 0;               // ring position / phase kept as counters: no divisions on the issue paths
      const int units = *p.n_rows * p.H * p.QT;
      int2 ent = attn_row_entry((int)blockIdx.x, units, p);
      for (int u = blockIdx.x; u < units; u += (int)gridDim.x, ++uc) {
        const int2 ent_next = attn_row_entry(u + (int)gridDim.x, units, p);
        const int br = ent.x, n_kt = min(ent.y, p.n_kt);
        const int qt = u % p.QT, h = (u / p.QT) % p.H;
        const int b = br / p.R;
        const int i0 = qt * AT_BQ;
        const uint32_t qb = uc & 1;
        tc::mbar_wait(&q_empty[qb], ((uc >> 1) & 1) ^ 1);
        tc::mbar_arrive_expect_tx(&q_full[qb], SM::Q_BYTES);
        uint8_t* qs = smem + SM::Q_OFF + qb * SM::Q_BYTES;
        tc::tma_load_3d(qs, &tmQK, &q_full[qb], h * 32, i0, br);            // box {32, 64, 1} twice: rows i0.., i0+64..
        tc::tma_load_3d(qs + 64 * 64, &tmQK, &q_full[qb], h * 32, i0 + 64, br);
        for (int kt = 0; kt < n_kt; ++kt) {
          tc::mbar_wait(&kv_empty[s], sph ^ 1);
          uint8_t* st = smem + SM::STAGE_OFF + s * p.stage_bytes;
          tc::mbar_arrive_expect_tx(&kv_full[s], stage_tx);
          tc::tma_load_3d(st, &tmQK, &kv_full[s], C + h * 32, kt * AT_BK, br);
          tc::tma_load_2d(st + SM::K_BYTES, &tmV, &kv_full[s], kt * AT_BK, (br * p.H + h) * 32);
          if (p.has_bias) tc::tma_load_3d(st + SM::K_BYTES + SM::V_BYTES, &tmBias, &kv_full[s], kt * AT_BK, i0, b * p.H + h);
          if (++s == (uint32_t)ST) { s = 0; sph ^= 1; }
        }
        ent = ent_next;
      }
    }
  } else if (warp == 5) {
    // ============================================================= MMA issue
    if (tc::elect_one()) {
      constexpr uint32_t idesc_s = tc::idesc_bf16_f32(AT_BQ, AT_BK);
      constexpr uint32_t idesc_b = tc::idesc_f16_f32(AT_BQ, AT_BK);   // bias tile x identity: fp16 operands
      constexpr uint32_t idesc_o = tc::idesc_bf16_f32(AT_BQ, 32);
      const uint64_t id_desc = tc::smem_desc_kmajor<128>(tc::smem_u32(smem + SM::ID_OFF));
      // issue side: S(j) = Q K^T for the next (unit, key tile); consume side: P(i) V.  j runs one step ahead of i.
      const int units = *p.n_rows * p.H * p.QT;
      int cu = blockIdx.x, ckt = 0;
      int2 ent = attn_row_entry(cu, units, p), ent_next = make_int2(0, 0);
      int cn = min(ent.y, p.n_kt);
      uint32_t cuc = 0, j = 0, i = 0;
      uint32_t js = 0, jph = 0, is = 0;              // ring position / phase of the issue side (j) and position of the consume side (i)
      // consume side: which key tile of its unit step i is (O accumulates in TMEM over the key tiles of a unit)
      int pu = blockIdx.x, pkt = 0, pn = cn;
      auto issue_s = [&]() -> bool {
        if (cu >= units) return false;
        const uint32_t qb = cuc & 1, s = js;
        if (ckt == 0) {
          ent_next = attn_row_entry(cu + (int)gridDim.x, units, p);   // used when this unit's last S has been issued
          tc::mbar_wait(&q_full[qb], (cuc >> 1) & 1);
        }
        tc::mbar_wait(&kv_full[s], jph);
        tc::tc_fence_after();
        const uint64_t q_desc = tc::smem_desc_kmajor<64>(tc::smem_u32(smem + SM::Q_OFF + qb * SM::Q_BYTES));
        const uint64_t k_desc = tc::smem_desc_kmajor<64>(tc::smem_u32(smem + SM::STAGE_OFF + s * p.stage_bytes));
        const uint32_t d = tmem_S + (j & 1) * AT_BK;
        tc::mma_bf16(d, q_desc, k_desc, idesc_s, false);
        tc::mma_bf16(d, q_desc + 2, k_desc + 2, idesc_s, true);
        if (p.has_bias) {   // S += bias I: the pair-bias tile of this stage as A operand, the identity as B
          const uint64_t b_desc = tc::smem_desc_kmajor<128>(
              tc::smem_u32(smem + SM::STAGE_OFF + s * p.stage_bytes + SM::K_BYTES + SM::V_BYTES));
#pragma unroll
          for (int k = 0; k < AT_BK / 16; ++k) tc::mma_bf16(d, b_desc + 2 * k, id_desc + 2 * k, idesc_b, true);
        }
        tc::mma_commit(&s_full[j & 1]);
        if (ckt == cn - 1) {
          tc::mma_commit(&q_empty[qb]);
          cu += (int)gridDim.x;
          cn = min(ent_next.y, p.n_kt);
          ckt = 0;
          ++cuc;
        } else {
          ++ckt;
        }
        ++j;
        if (++js == (uint32_t)ST) { js = 0; jph ^= 1; }
        return true;
      };
      if (issue_s()) {
        while (true) {
          issue_s();                               // S(i-1) was drained before P(i-1) arrived, so its buffer is free
          const uint32_t s = is;
          if (++is == (uint32_t)ST) is = 0;
          tc::mbar_wait(p_full, i & 1);
          tc::tc_fence_after();
          const uint64_t v_desc = tc::smem_desc_kmajor<128>(tc::smem_u32(smem + SM::STAGE_OFF + s * p.stage_bytes + SM::K_BYTES));
#pragma unroll
          for (int k = 0; k < AT_BK / 16; ++k)   // A = P(i): bf16 pairs in the first 32 columns of the S buffer it came from
            tc::mma_bf16_ts(tmem_O, tmem_S + (i & 1) * AT_BK + k * 8, v_desc + 2 * k, idesc_o, (k | pkt) != 0);
          tc::mma_commit(o_full);
          tc::mma_commit(&kv_empty[s]);
          if (++pkt == pn) {
            pu += (int)gridDim.x;
            pn = min(attn_row_entry(pu, units, p).y, p.n_kt);
            pkt = 0;
          }
          if (++i == j) break;
        }
      }
    }
  } else {
    // ============================================================= softmax warps (thread per query row)
    const int row = warp * 32 + lane;            // warp w reads TMEM lanes [32w, 32w+32)
    const uint32_t lane_addr = (uint32_t)(warp * 32) << 16;
    int cur_b = -1;
    uint32_t tile_masked = 0;                    // bit kt: key tile kt holds a masked / out-of-range key
    uint32_t i = 0;                              // pipeline step (all units)
    const int units = *p.n_rows * p.H * p.QT;
    // unit u = (row entry ridx, head h, query tile qt): advanced incrementally (the integer divisions of the direct form are
    // long dependent chains through the unit that is busy with the exponentials: ~0.4 us per unit on this critical path)
    const int G = (int)gridDim.x;
    const int g_qt = G % p.QT, g_h = (G / p.QT) % p.H, g_r = G / (p.QT * p.H);
    int qt = (int)blockIdx.x % p.QT, h = ((int)blockIdx.x / p.QT) % p.H, ridx = (int)blockIdx.x / (p.QT * p.H);
    int2 ent = (int)blockIdx.x < units ? __ldg(p.rows + ridx) : make_int2(0, 0);
    for (int u = blockIdx.x; u < units; u += G) {
      // next unit's coordinates and row entry (a plain load, used one unit later)
      int nqt = qt + g_qt, nh = h + g_h, nr = ridx + g_r;
      if (nqt >= p.QT) { nqt -= p.QT; ++nh; }
      if (nh >= p.H) { nh -= p.H; ++nr; }
      const int2 ent_next = u + G < units ? __ldg(p.rows + nr) : make_int2(0, 0);
      const int br = ent.x, n_kt = min(ent.y, p.n_kt);
      const int b = br / p.R;
      const int qi = qt * AT_BQ + row;
      if (b != cur_b) {
        // key mask of this protein as one bit per key (1 = masked or out of range, R3) + one bit per key tile
        tc::named_bar_sync(1, 128);
        if (threadIdx.x == 0) *maskbits = 0;
        tc::named_bar_sync(1, 128);
        for (int j = threadIdx.x; j < p.n_kt * AT_BK; j += 128) {
          const bool keep = j < p.L && p.keymask[(long)b * p.L + j] > 0.5f;
          const uint32_t w = __ballot_sync(0xffffffffu, !keep);
          if (lane == 0) {
            mbits[j >> 5] = w;
            if (w) atomicOr(maskbits, 1u << (j / AT_BK));
          }
        }
        tc::named_bar_sync(1, 128);
        tile_masked = *maskbits;
        cur_b = b;
      }
      // the gate of this row (fp16, bounded in [0,1], not an MMA operand): fetched now, used after the last key tile
      uint4 gq[4];
      if (qi < p.L) {
        const uint4* gp = reinterpret_cast<const uint4*>(p.qkg + ((long)br * p.L + qi) * (3 * C) + 2 * C + h * 32);
#pragma unroll
        for (int d = 0; d < 4; ++d) gq[d] = __ldg(gp + d);
      } else {
#pragma unroll
        for (int d = 0; d < 4; ++d) gq[d] = make_uint4(0u, 0u, 0u, 0u);
      }
      // Online softmax with the output accumulated by the tensor core: O stays in TMEM over the key tiles of the unit
      // (P V with accumulate) and P is taken relative to a reference maximum m_ref that is only moved when the running
      // maximum has grown by more than 2^8 beyond it (P <= 256 then, exact in the exp2 domain: the common factor cancels in
      // O / l).  Moving it rescales O in TMEM (load, multiply, store) and l; after the first tiles of a row that is rare, so
      // the per-tile "O = (O + PV) alpha" round trip through registers is gone.
      float m_run = -INFINITY, m_ref = -INFINITY, l_run = 0.f;
      for (int kt = 0; kt < n_kt; ++kt, ++i) {
        tc::mbar_wait(&s_full[i & 1], (i >> 1) & 1);
        tc::tc_fence_after();
        uint32_t sv[2][32];
        tc::tmem_ld32(tmem_S + lane_addr + (i & 1) * AT_BK, sv[0]);
        tc::tmem_ld32(tmem_S + lane_addr + (i & 1) * AT_BK + 32, sv[1]);
        tc::tmem_ld_wait();
        float x[64];   // logits in the exp2 domain; the pair bias was already added by the tensor core
#pragma unroll
        for (int j = 0; j < 64; ++j) x[j] = __uint_as_float(sv[j >> 5][j & 31]);
        if ((tile_masked >> kt) & 1) {
          const uint32_t w0 = mbits[2 * kt], w1 = mbits[2 * kt + 1];
#pragma unroll
          for (int j = 0; j < 32; ++j) {
            if ((w0 >> j) & 1) x[j] = -INFINITY;
            if ((w1 >> j) & 1) x[32 + j] = -INFINITY;
          }
        }
        float mx0 = x[0], mx1 = x[1], mx2 = x[2], mx3 = x[3];
#pragma unroll
        for (int j = 4; j < 64; j += 4) {
          mx0 = fmaxf(mx0, x[j]);
          mx1 = fmaxf(mx1, x[j + 1]);
          mx2 = fmaxf(mx2, x[j + 2]);
          mx3 = fmaxf(mx3, x[j + 3]);
        }
        m_run = fmaxf(m_run, fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)));
        bool pv_seen = (kt == 0);   // PV(i-1) observed complete (the previous unit's last one was, at that unit's end)
        if (kt == 0) {
          m_ref = m_run;
        } else {
          const bool move = m_run > m_ref + 8.0f;          // also true when m_ref is still -inf and a key has appeared
          if (__any_sync(0xffffffffu, move)) {
            // PV(i-1) must have finished before O is touched
            tc::mbar_wait(o_full, (i - 1) & 1);
            tc::tc_fence_after();
            pv_seen = true;
            // rows that do not move multiply by 1; a row whose reference was -inf has O = l = 0: factor 0 keeps that exact
            const float alpha = !move ? 1.0f : (m_ref == -INFINITY ? 0.0f : ex2_approx(m_ref - m_run));
            uint32_t ov[32];
            tc::tmem_ld32(tmem_O + lane_addr, ov);
            tc::tmem_ld_wait();
#pragma unroll
            for (int d = 0; d < 32; ++d) ov[d] = __float_as_uint(__uint_as_float(ov[d]) * alpha);
            tc::tmem_st32(tmem_O + lane_addr, ov);
            tc::tmem_st_wait();
            l_run *= alpha;
            if (move) m_ref = m_run;
          }
        }
        const float m_use = (m_ref == -INFINITY) ? 0.f : m_ref;
        float sum0 = 0.f, sum1 = 0.f;
        uint32_t pk[32];
#pragma unroll
        for (int e = 0; e < 32; ++e) {
          const float p0 = ex2_approx(x[2 * e] - m_use), p1 = ex2_approx(x[2 * e + 1] - m_use);
          sum0 += p0;
          sum1 += p1;
          __nv_bfloat162 pp = __floats2bfloat162_rn(p0, p1);
          pk[e] = *reinterpret_cast<uint32_t*>(&pp);
        }
        l_run += sum0 + sum1;
        // Steps that did not rescale wait for PV(i-1) only here, after the exponentials (P(i) goes into the buffer S(i) came
        // from, not the one PV(i-1) reads, so nothing above depended on it).  The wait itself must not be dropped: a one-bit
        // phase parity is only unambiguous while this thread has seen every phase but the newest, and PV(i) cannot complete
        // before the arrival below.
        if (!pv_seen) tc::mbar_wait(o_full, (i - 1) & 1);
        // P(i) stays in tensor memory: bf16 pairs over the first 32 columns of this thread's own (already loaded) logits
        tc::tmem_st32(tmem_S + lane_addr + (i & 1) * AT_BK, pk);
        tc::tmem_st_wait();
        tc::tc_fence_before();
        tc::mbar_arrive(p_full);
      }
      // the unit's O (all key tiles, relative to m_ref), then normalise, gate and store this row's 32 output channels
      tc::mbar_wait(o_full, (i - 1) & 1);
      tc::tc_fence_after();
      float oacc[32];
      {
        uint32_t ov[32];
        tc::tmem_ld32(tmem_O + lane_addr, ov);
        tc::tmem_ld_wait();
#pragma unroll
        for (int d = 0; d < 32; ++d) oacc[d] = __uint_as_float(ov[d]);
      }
      tc::tc_fence_before();
      if (qi < p.L) {
        const float inv = l_run > 0.f ? 1.0f / l_run : 0.f;
        bf16* op = p.o + ((long)br * p.L + qi) * C + h * 32;
#pragma unroll
        for (int d = 0; d < 4; ++d) {
          const uint32_t gw[4] = {gq[d].x, gq[d].y, gq[d].z, gq[d].w};
          uint32_t pk[4];
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const __half2 g2 = *reinterpret_cast<const __half2*>(&gw[e]);
            __nv_bfloat162 pp = __floats2bfloat162_rn(oacc[d * 8 + 2 * e] * inv * __low2float(g2),
                                                      oacc[d * 8 + 2 * e + 1] * inv * __high2float(g2));
            pk[e] = *reinterpret_cast<uint32_t*>(&pp);
          }
          *reinterpret_cast<uint4*>(op + d * 8) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
        }
      }
      ent = ent_next;
      qt = nqt; h = nh; ridx = nr;
    }
  }
  tc::tc_fence_before();
  __syncthreads();
  if (warp == 5) tc::tmem_dealloc<256>(tmem_base);
}

bool configure_attn_kernel() {
  cudaError_t e = cudaFuncSetAttribute(attn_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, AttnSmem::TOTAL);
  if (e != cudaSuccess) tc_set_error(std::string("cudaFuncSetAttribute(attn_tc): ") + cudaGetErrorString(e));
  return e == cudaSuccess;
}

int launch_attn_tc(TmaCtx* ctx, const bf16* qkg, const bf16* vt, const bf16* bias, const float* keymask, bf16* o, int B,
                   int R, int L, int Lpad, int H, const void* rows, const int* n_rows, int num_sms, cudaStream_t st) {
  if (L > AT_MAXKEYS) {
    tc_set_error("attn_tc: key length above 1024 not supported");
    return -1;
  }
  const int C = H * 32;
  CUtensorMap tmQK, tmV, tmB;
  {
    uint64_t d[3] = {(uint64_t)3 * C, (uint64_t)L, (uint64_t)B * R}, s[2] = {(uint64_t)3 * C, (uint64_t)L * 3 * C};
    uint32_t bx[3] = {32, 64, 1};
    if (tma_encode_bf16(ctx, &tmQK, qkg, 3, d, s, bx, 64) != 0) return -1;
  }
  {
    uint64_t d[2] = {(uint64_t)L, (uint64_t)B * R * H * 32}, s[1] = {(uint64_t)Lpad};
    uint32_t bx[2] = {64, 32};
    if (tma_encode_bf16(ctx, &tmV, vt, 2, d, s, bx, 128) != 0) return -1;
  }
  if (bias) {
    uint64_t d[3] = {(uint64_t)L, (uint64_t)L, (uint64_t)B * H}, s[2] = {(uint64_t)Lpad, (uint64_t)L * Lpad};
    uint32_t bx[3] = {64, 128, 1};
    if (tma_encode_bf16(ctx, &tmB, bias, 3, d, s, bx, 128) != 0) return -1;
  } else {
    tmB = tmV;
  }
  AttnParams p;
  p.qkg = qkg; p.keymask = keymask; p.o = o;
  p.R = R; p.L = L; p.H = H;
  p.QT = (L + AT_BQ - 1) / AT_BQ;
  p.n_kt = (L + AT_BK - 1) / AT_BK;
  p.has_bias = bias ? 1 : 0;
  p.stage_bytes = AttnSmem::K_BYTES + AttnSmem::V_BYTES + (bias ? AttnSmem::B_BYTES : 0);
  p.stages = bias ? 3 : AttnSmem::MAX_STAGES;
  const long units = (long)B * R * H * p.QT;      // upper bound (all rows active)
  if (units >= (1L << 31) - 4096) {
    tc_set_error("attn_tc: too many work units");
    return -1;
  }
  p.rows = reinterpret_cast<const int2*>(rows);
  p.n_rows = n_rows;
  const long max_ctas = 2L * num_sms;
  unsigned grid = (unsigned)(units < max_ctas ? units : max_ctas);
  attn_tc_kernel<<<grid, AT_THREADS, AttnSmem::TOTAL, st>>>(tmQK, tmV, tmB, p);
  return 0;
}

}  // namespace pf
