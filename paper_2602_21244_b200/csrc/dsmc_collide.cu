// Fused neural DSMC collision step: chi-table variant and FP32 CUDA-core MLP variants.
// (The BF16 tcgen05 variant lives in dsmc_collide_tc.cu; all share dsmc_chunk.cuh.)
//
// One CTA owns one chunk (dsmc_chunk.cuh): 12 B read + 12 B write per particle, everything else
// on chip.  Chunks that do not fit the small shared-memory footprint (a cell above ~1000 particles,
// or more than 64 non-trivial cells in 512 slots) are appended to a deferred list and processed by
// a second, larger-footprint launch of the same code.
#include <algorithm>

#include "dsmc_chunk.cuh"

namespace dsmc {

// k_chunk_map: chunk_first[b] = first cell whose first slot is >= b * kChunk; resets the deferred list.
__global__ void k_chunk_map(int32_t K, const int32_t *__restrict__ cs, int32_t *__restrict__ chunk_first,
                            int32_t *__restrict__ big, int32_t *__restrict__ big2, int32_t *__restrict__ work) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k == 0) {
    big[0] = 0;
    big2[0] = 0;
    work[0] = 0;
    work[1] = 0;
    work[2] = 0;
  }
  if (k > K) return;
  const int s = __ldg(cs + k);
  const int lo = (k == 0) ? 0 : (__ldg(cs + k - 1) / kChunk + 1);
  const int hi = s / kChunk;
  for (int b = lo; b <= hi; ++b) chunk_first[b] = k;
}

// k_chunk_meta: (first cell, end cell, first slot, end slot) of every chunk, so a CTA starts with one load
__global__ void k_chunk_meta(int32_t n_chunks, int32_t K, const int32_t *__restrict__ cs,
                             const int32_t *__restrict__ chunk_first, int4 *__restrict__ meta) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= n_chunks) return;
  const int c_lo = chunk_first[b], c_hi = (b + 1 < n_chunks) ? chunk_first[b + 1] : K;
  meta[b] = make_int4(c_lo, c_hi, __ldg(cs + min(c_lo, K)), __ldg(cs + min(c_hi, K)));
}

// ---------------------------------------------------------------------------------------------
// FP32 MLP over a tile of TP pairs.  X = buf[0] holds features [k][TP]; result left in the
// returned buffer as [o][TP].  Thread (tp = tid % (TP/4), to = tid / (TP/4)) owns 4 pairs x
// outputs {to, to + n_to, ...}.
// ---------------------------------------------------------------------------------------------
template <int TP>
__device__ float *mlp_tile_fp32(const MlpDev &net, float *buf) {
  constexpr int NTP = TP / 4, NTO = kThreads / NTP, MAXM = 256 / NTO > 8 ? 8 : 256 / NTO;
  const int tid = threadIdx.x, tp = tid % NTP, to = tid / NTP;
  float *in = buf, *out = buf + net.dmax * TP;
  for (int l = 0; l < net.n_layers; ++l) {
    const int Din = net.dims[l], Dout = net.dims[l + 1];
    const float *__restrict__ Wt = net.Wt[l];
    const bool hidden = (l + 1 < net.n_layers);
    for (int m0 = 0; m0 * NTO < Dout; m0 += MAXM) {
      float acc[MAXM][4];
#pragma unroll
      for (int m = 0; m < MAXM; ++m) {
        const int o = to + NTO * (m0 + m);
        const float b = o < Dout ? __ldg(net.b[l] + o) : 0.f;
        acc[m][0] = b; acc[m][1] = b; acc[m][2] = b; acc[m][3] = b;
      }
      for (int k = 0; k < Din; ++k) {
        const float4 x = *reinterpret_cast<const float4 *>(in + k * TP + 4 * tp);
#pragma unroll
        for (int m = 0; m < MAXM; ++m) {
          const int o = to + NTO * (m0 + m);
          if (NTO * (m0 + m) < Dout) {  // CTA-uniform
            const float w = o < Dout ? __ldg(Wt + k * Dout + o) : 0.f;
            acc[m][0] = fmaf(w, x.x, acc[m][0]);
            acc[m][1] = fmaf(w, x.y, acc[m][1]);
            acc[m][2] = fmaf(w, x.z, acc[m][2]);
            acc[m][3] = fmaf(w, x.w, acc[m][3]);
          }
        }
      }
#pragma unroll
      for (int m = 0; m < MAXM; ++m) {
        const int o = to + NTO * (m0 + m);
        if (o < Dout) {
          float4 y;
          y.x = hidden ? act_apply(net.act, acc[m][0]) : acc[m][0];
          y.y = hidden ? act_apply(net.act, acc[m][1]) : acc[m][1];
          y.z = hidden ? act_apply(net.act, acc[m][2]) : acc[m][2];
          y.w = hidden ? act_apply(net.act, acc[m][3]) : acc[m][3];
          *reinterpret_cast<float4 *>(out + o * TP + 4 * tp) = y;
        }
      }
    }
    __syncthreads();
    float *t = in; in = out; out = t;
  }
  return in;
}


// ---------------------------------------------------------------------------------------------
// pair phases
// ---------------------------------------------------------------------------------------------
template <class TM, class CK>
__device__ __forceinline__ void pairs_table(const TM &T, const StepParams &P, CK &S, int q0) {
  const int n_pairs = S.misc[MI_NPAIRS];
  const float nBm1 = (float)(P.table.nB - 1);
  const int stage = P.split_stage;
  for (int t = T.tid; t < n_pairs; t += TM::kN) {
    PairCtx c = pair_setup(P, S, t, true);
    float px = c.gx, py = c.gy, pz = c.gz, chi = 0.f;
    float sb;  // b~ = sqrt(U_b)
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(sb) : "f"(c.U_b));
    // split form of the chi-MLP step (launch_collide_replace_split): pair index = first slot of the cell / 2 + pair slot
    const int64_t pidx = ((int64_t)(q0 + c.start) >> 1) + c.s;
    if (stage == 3) {  // network inputs only (Q15): ((E~ - E~min) / (E~max - E~min) clamped to [0, 1], b~)
      const float e = (0.6931471806f * __log2f(P.e_coef * c.g2) - P.lnE_min) * P.inv_lnE_range;
      P.feat0[pidx] = !(e > 0.f) ? 0.f : fminf(e, 1.f);
      P.feat1[pidx] = sb;
      continue;
    }
    if (c.acc) {
      // E~ = ln(m g^2 / (4 kB))
      chi = stage == 4 ? __ldg(P.chi_pair + pidx) : chi_table_t(P.table, table_tE(P.table, P.e_coef * c.g2), sb * nBm1);
      if (c.g2 > 0.f) rotate_fast(c, chi, c.U_eps, px, py, pz);
    }
    pair_commit(P, S, c, px, py, pz, chi, q0);
  }
}

template <int TP, class CK>
__device__ __forceinline__ void pairs_mlp_fp32(const StepParams &P, const MlpDev &net, CK &S, float *mlp, int q0) {
  const int tid = threadIdx.x;
  const int n_pairs = S.misc[MI_NPAIRS];
  const int d0 = net.dims[0];
  for (int t0 = 0; t0 < n_pairs; t0 += TP) {
    PairCtx c;
    const bool mine = tid < TP && t0 + tid < n_pairs;
    if (tid < TP) {
      float x[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
      if (mine) {
        c = pair_setup(P, S, t0 + tid, P.op != 0);
        const CellInfo &ci = S.cells[c.a];
        if (P.op == 0) {  // VHS-NN features (eqs. 1-3, Q1-Q3)
          float n0 = 0.f, n1 = 0.f, n2 = 0.f;
          if (P.flags & DSMC_F_NOISE) {
            const uint4 r = philox4x32_10((uint32_t)c.s, c.cell + P.cell_base, P.step, 2u, P.seed_lo, P.seed_hi);
            box_muller3(r, n0, n1, n2);
            n0 *= P.noise_sigma; n1 *= P.noise_sigma; n2 *= P.noise_sigma;
          }
          x[0] = c.gx * P.inv_sigma_v; x[1] = c.gy * P.inv_sigma_v; x[2] = c.gz * P.inv_sigma_v;
          if (d0 == 8) {
            x[3] = sqrtf(c.g2) * P.inv_sigma_v;
            x[4] = ci.theta * P.T_coef / (float)ci.N * P.inv_T_scale;  // T = m Theta / (3 kB N)
            x[5] = n0; x[6] = n1; x[7] = n2;
          } else {
            x[3] = n0; x[4] = n1; x[5] = n2;
          }
        } else {  // chi-MLP inputs (Q15)
          const float lnE = logf(P.e_coef * c.g2);
          float e = (lnE - P.lnE_min) * P.inv_lnE_range;
          x[0] = !(e > 0.f) ? 0.f : fminf(e, 1.f);
          x[1] = sqrtf(c.U_b);
        }
      }
      for (int k = 0; k < d0; ++k) mlp[k * TP + tid] = x[k];
    }
    __syncthreads();
    const float *out = mlp_tile_fp32<TP>(net, mlp);
    if (mine) {
      float px = c.gx, py = c.gy, pz = c.gz, aux = 0.f;
      if (c.acc) {
        if (P.op == 0) {
          const float hx = out[tid], hy = out[TP + tid], hz = out[2 * TP + tid];
          const float hn = sqrtf(hx * hx + hy * hy + hz * hz);
          aux = hn;
          if (P.flags & DSMC_F_ENERGY_SHELL) {
            if (hn >= P.shell_eps) {  // eq. 5 with the guard of Q4
              const float sc = sqrtf(c.g2) / hn;
              px = sc * hx; py = sc * hy; pz = sc * hz;
            }
          } else {
            px = P.sigma_v * hx; py = P.sigma_v * hy; pz = P.sigma_v * hz;
          }
        } else {
          const float z = out[tid];
          const float y = fmaxf(z, 0.f) + log1pf(expf(-fabsf(z)));  // softplus
          aux = expm1f(y);                                           // chi
          if (c.g2 > 0.f) rotate_fast(c, aux, c.U_eps, px, py, pz);
        }
      }
      pair_commit(P, S, c, px, py, pz, aux, q0);
    }
    __syncthreads();
  }
}

// ---------------------------------------------------------------------------------------------
// kernels.  OP_TABLE: chi-table operator; otherwise FP32 MLP (P.op = 0 VHS-NN, 2 chi-MLP).
// DEFERRED: persistent loop over the deferred chunk list instead of chunk = blockIdx.x.
// ---------------------------------------------------------------------------------------------
// SRC: where a CTA's chunks come from (0 = chunk blockIdx.x, 1 = deferred list P.big, 2 = second list P.big2,
// walked grid-stride).  DST: where a chunk that does not fit this footprint goes (1 = P.big, 2 = P.big2,
// 0 = nowhere: DSMC_ERR_CELL_TOO_LARGE).
template <int NT, class CK, bool OP_TABLE, int TP, int DST>
__device__ __forceinline__ void process_chunk(const StepParams &P, const MlpDev &net, CK &S, float *mlp, int chunk) {
  const TeamT<NT> T{(int)threadIdx.x, 0};
  int q0 = 0;
  const int n_loc = chunk_begin(T, P, S, chunk, q0);
  if (n_loc == 0) return;
  if (n_loc < 0) {
    if (threadIdx.x == 0) {
      if (DST == 0) {
        *P.status = DSMC_ERR_CELL_TOO_LARGE;
      } else {
        int32_t *list = DST == 1 ? P.big : P.big2;
        const int i = atomicAdd(list, 1);
        list[1 + i] = chunk;
      }
    }
    return;
  }
  chunk_pre_and_sort(T, P, S, n_loc);
  if (OP_TABLE) {
    pairs_table(T, P, S, q0);
    if (P.split_stage == 3) return;  // (uniform) first pass of the split form: nothing committed, nothing to store
  } else {
    pairs_mlp_fp32<TP>(P, net, S, mlp, q0);
  }
  T.sync();
  chunk_finish(T, P, S, n_loc, q0);
}

template <int LMAX, int AMAX, bool OP_TABLE, int TP, int SRC, int DST, int MINB, int NT = kThreads, bool REPL = false>
__global__ void __launch_bounds__(NT, MINB) k_collide(const StepParams P, const MlpDev net) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Chunk<LMAX, AMAX, REPL, OP_TABLE> S;
  float *mlp = reinterpret_cast<float *>(S.carve(smem_raw));
  if (SRC == 0) {
    process_chunk<NT, Chunk<LMAX, AMAX, REPL, OP_TABLE>, OP_TABLE, TP, DST>(P, net, S, mlp, blockIdx.x);
  } else {
    const int32_t *list = SRC == 1 ? P.big : P.big2;
    const int n_list = *reinterpret_cast<volatile const int32_t *>(list);
    for (int i = blockIdx.x; i < n_list; i += gridDim.x) {
      process_chunk<NT, Chunk<LMAX, AMAX, REPL, OP_TABLE>, OP_TABLE, TP, DST>(P, net, S, mlp, list[1 + i]);
      __syncthreads();
    }
  }
}

template <int LMAX, int AMAX, bool OP_TABLE, int TP, int SRC, int DST, int MINB, int NT = kThreads, bool REPL = false>
static int launch_one(dsmc_ctx *c, const StepParams &p, const MlpDev &nd, int grid, size_t mlp_bytes) {
  auto kern = k_collide<LMAX, AMAX, OP_TABLE, TP, SRC, DST, MINB, NT, REPL>;
  const size_t smem = Chunk<LMAX, AMAX>::bytes() + mlp_bytes;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return DSMC_ERR_CUDA;
  kern<<<grid, NT, smem, c->stream>>>(p, nd);
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

int launch_chunk_map(dsmc_ctx *c, StepParams &p) {
  p.n_chunks = (int32_t)((p.n + kChunk - 1) / kChunk);
  p.chunk_first = c->d_chunk_first;
  p.big = c->d_big;
  p.big2 = c->d_big2;
  p.work = c->d_work;
  k_chunk_map<<<(p.n_cells + 1 + 255) / 256, 256, 0, c->stream>>>(p.n_cells, p.cell_start, c->d_chunk_first, c->d_big,
                                                                  c->d_big2, c->d_work);
  p.chunk_meta = c->d_chunk_meta;
  k_chunk_meta<<<(p.n_chunks + 255) / 256, 256, 0, c->stream>>>(p.n_chunks, p.n_cells, p.cell_start, c->d_chunk_first,
                                                             c->d_chunk_meta);
  c->launches += 2;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

// ---------------------------------------------------------------------------------------------
// VHS-NN operator on the tensor cores with pairs drawn WITH replacement (DSMC_F_PAIR_REPLACE | DSMC_F_BF16_TC): the
// split form on the with-replacement chunk machinery.  Pass 1: draw the pairs, network inputs of every pair (eqs. 1-3)
// -> pair arrays.  Pass 2: k_mlp_rows_tc_split (dsmc_collide_tc.cu).  Pass 3: draw the same pairs again, outputs ->
// eq. 5 -> changes added up per particle (batch semantics, Q29), moment matching, store.  (Without replacement the
// split form runs on the cell-team kernels, dsmc_cells.cu.)
// ---------------------------------------------------------------------------------------------
template <class TM, class CK>
__device__ __forceinline__ void pairs_vhs_split(const TM &T, const StepParams &P, CK &S, int q0) {
  const int n_pairs = S.misc[MI_NPAIRS];
  const int stage = P.split_stage, d_in = P.split_din;
  const int64_t np = P.split_np;
  for (int t = T.tid; t < n_pairs; t += TM::kN) {
    PairCtx c = pair_setup(P, S, t, false);
    const int64_t pidx = ((int64_t)(q0 + c.start) >> 1) + c.s;
    if (stage == 3) {  // VHS-NN features (eqs. 1-3, Q1-Q3)
      float x[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
      float n0 = 0.f, n1 = 0.f, n2 = 0.f;
      if (P.flags & DSMC_F_NOISE) {
        const uint4 r = philox4x32_10((uint32_t)c.s, c.cell + P.cell_base, P.step, 2u, P.seed_lo, P.seed_hi);
        box_muller3(r, n0, n1, n2);
        n0 *= P.noise_sigma; n1 *= P.noise_sigma; n2 *= P.noise_sigma;
      }
      x[0] = c.gx * P.inv_sigma_v; x[1] = c.gy * P.inv_sigma_v; x[2] = c.gz * P.inv_sigma_v;
      if (d_in == 8) {
        const CellInfo &ci = S.cells[c.a];
        x[3] = sqrtf(c.g2) * P.inv_sigma_v;
        x[4] = ci.theta * P.T_coef / (float)ci.N * P.inv_T_scale;  // T = m Theta / (3 kB N)
        x[5] = n0; x[6] = n1; x[7] = n2;
      } else {
        x[3] = n0; x[4] = n1; x[5] = n2;
      }
#pragma unroll
      for (int k = 0; k < 8; ++k)
        if (k < d_in) P.feat0[k * np + pidx] = x[k];
      continue;
    }
    float px = c.gx, py = c.gy, pz = c.gz, aux = 0.f;
    if (c.acc) {
      const float hx = __ldg(P.out3[0] + pidx), hy = __ldg(P.out3[1] + pidx), hz = __ldg(P.out3[2] + pidx);
      const float hn = sqrtf(hx * hx + hy * hy + hz * hz);
      aux = hn;
      if (P.flags & DSMC_F_ENERGY_SHELL) {
        if (hn >= P.shell_eps) {  // eq. 5 with the guard of Q4
          const float sc = sqrtf(c.g2) / hn;
          px = sc * hx; py = sc * hy; pz = sc * hz;
        }
      } else {
        px = P.sigma_v * hx; py = P.sigma_v * hy; pz = P.sigma_v * hz;
      }
    }
    pair_commit(P, S, c, px, py, pz, aux, q0);
  }
}

template <int LMAX, int AMAX, int SRC, int DST, int MINB>
__global__ void __launch_bounds__(kThreads, MINB) k_vhs_replace_split(const StepParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  using CK = Chunk<LMAX, AMAX, true, false>;
  CK S;
  S.carve(smem_raw);
  const TeamT<kThreads> T{(int)threadIdx.x, 0};
  auto one = [&](int chunk) {
    int q0 = 0;
    const int n_loc = chunk_begin(T, P, S, chunk, q0);
    if (n_loc == 0) return;
    if (n_loc < 0) {
      if (threadIdx.x == 0) {
        if (DST == 0) {
          *P.status = DSMC_ERR_CELL_TOO_LARGE;
        } else {
          const int i = atomicAdd(P.big, 1);
          P.big[1 + i] = chunk;
        }
      }
      return;
    }
    chunk_pre_and_sort(T, P, S, n_loc);
    pairs_vhs_split(T, P, S, q0);
    if (P.split_stage == 3) return;
    T.sync();
    chunk_finish(T, P, S, n_loc, q0);
  };
  if (SRC == 0) {
    one(blockIdx.x);
  } else {
    const int n_list = *reinterpret_cast<volatile const int32_t *>(P.big);
    for (int i = blockIdx.x; i < n_list; i += gridDim.x) {
      one(P.big[1 + i]);
      __syncthreads();
    }
  }
}

template <int LMAX, int AMAX, int SRC, int DST, int MINB>
static int launch_vhs_replace_split_one(dsmc_ctx *c, const StepParams &p, int grid) {
  auto kern = k_vhs_replace_split<LMAX, AMAX, SRC, DST, MINB>;
  const size_t smem = Chunk<LMAX, AMAX>::bytes();
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return DSMC_ERR_CUDA;
  kern<<<grid, kThreads, smem, c->stream>>>(p);
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

int launch_collide_vhs_replace_split(dsmc_ctx *c, const StepParams &p_in, const MlpTcDev *net) {
  const TcTailF32 *tail = &c->tc_tail[0];
  if (p_in.op != 0 || !((net->d_in == 8 || net->d_in == 6) && net->d_out == 3) || tail->d_out != 3)
    return DSMC_ERR_UNSUPPORTED_SHAPE;
  StepParams p = p_in;
  const int64_t np = (p.n / 2 + 4) & ~(int64_t)3;
  p.feat0 = reinterpret_cast<float *>(c->d_bin_rec[0]);  // 8 arrays of np floats: 16 B / particle + 128 B
  p.split_np = np;
  p.split_din = net->d_in;
  p.out3[0] = reinterpret_cast<float *>(c->d_bin_cell[0]);
  p.out3[1] = p.out3[0] + np;
  p.out3[2] = reinterpret_cast<float *>(c->d_bin_cell[1]);
  for (int stage = 3; stage <= 4; ++stage) {
    int rc = launch_chunk_map(c, p);  // (also resets the deferred-chunk list)
    if (rc != DSMC_OK) return rc;
    p.split_stage = stage;
    rc = launch_vhs_replace_split_one<kLmaxSmall, kAmaxSmall, 0, 1, 3>(c, p, p.n_chunks);
    if (rc != DSMC_OK) return rc;
    rc = launch_vhs_replace_split_one<kLmaxBig, kAmaxBig, 1, 0, 1>(c, p, c->num_sms);
    if (rc != DSMC_OK) return rc;
    if (stage == 3) {
      rc = launch_mlp_rows_tc_split(c, p.n / 2 + 1, p.feat0, np, p.out3[0], p.out3[1], p.out3[2], net, tail);
      if (rc != DSMC_OK) return rc;
    }
  }
  return DSMC_OK;
}

// chi-MLP on the tensor cores with pairs drawn WITH replacement (DSMC_F_PAIR_REPLACE | DSMC_F_BF16_TC): the split form
// of dsmc_cells.cu on the with-replacement chunk kernels.  Pass 1 draws the pairs and writes the two network inputs of
// every pair, pass 2 is k_chi_batch_tc on those arrays, pass 3 draws the same pairs again (counter-based randoms),
// rotates by the chi of pass 2, adds up the changes and matches.
static int launch_replace_table_kernels(dsmc_ctx *c, const StepParams &p) {
  MlpDev nd{};
  int rc = launch_one<704, 32, true, 64, 0, 1, 9, 128, true>(c, p, nd, p.n_chunks, 0);
  if (rc != DSMC_OK) return rc;
  rc = launch_one<1024, 8, true, 64, 1, 2, 7, 128, true>(c, p, nd, c->num_sms * 7, 0);
  if (rc != DSMC_OK) return rc;
  return launch_one<kLmaxBig, kAmaxBig, true, 64, 2, 0, 1, kThreads, true>(c, p, nd, c->num_sms, 0);
}

int launch_collide_replace_split(dsmc_ctx *c, const StepParams &p_in, const MlpTcDev *net) {
  if (p_in.op != 2 || net->d_in != 2 || net->d_out != 1 || (net->H != 64 && net->H != 128))
    return DSMC_ERR_UNSUPPORTED_SHAPE;
  StepParams p = p_in;
  const int64_t np = (p.n / 2 + 4) & ~(int64_t)3;
  float *base = reinterpret_cast<float *>(c->d_bin_rec[0]);
  p.feat0 = base;
  p.feat1 = base + np;
  p.chi_pair = base + 2 * np;
  int rc = launch_chunk_map(c, p);
  if (rc != DSMC_OK) return rc;
  p.split_stage = 3;
  rc = launch_replace_table_kernels(c, p);
  if (rc != DSMC_OK) return rc;
  rc = launch_chi_rows_tc(c, p.n / 2 + 1, p.feat0, p.feat1, p.chi_pair, net);
  if (rc != DSMC_OK) return rc;
  rc = launch_chunk_map(c, p);  // (resets the deferred-chunk lists and work counters)
  if (rc != DSMC_OK) return rc;
  p.split_stage = 4;
  return launch_replace_table_kernels(c, p);
}

int launch_collide(dsmc_ctx *c, const StepParams &p_in, const MlpDev *net) {
  if (p_in.op == 1 && !(p_in.flags & DSMC_F_PAIR_REPLACE)) return launch_collide_cells(c, p_in);  // dsmc_cells.cu
  StepParams p = p_in;
  int rc = launch_chunk_map(c, p);
  if (rc != DSMC_OK) return rc;
  MlpDev nd{};
  const int big_grid = c->num_sms;
  if (p.flags & DSMC_F_PAIR_REPLACE) {  // pairs drawn with replacement: separate instantiations
    if (p.op == 1) {
      rc = launch_one<704, 32, true, 64, 0, 1, 9, 128, true>(c, p, nd, p.n_chunks, 0);
      if (rc != DSMC_OK) return rc;
      rc = launch_one<1024, 8, true, 64, 1, 2, 7, 128, true>(c, p, nd, c->num_sms * 7, 0);
      if (rc != DSMC_OK) return rc;
      return launch_one<kLmaxBig, kAmaxBig, true, 64, 2, 0, 1, kThreads, true>(c, p, nd, big_grid, 0);
    }
    nd = *net;
    if (nd.dmax > 128) return DSMC_ERR_UNSUPPORTED_SHAPE;
    const size_t mbr = sizeof(float) * 2 * nd.dmax * 64;
    rc = launch_one<kLmaxSmall, kAmaxSmall, false, 64, 0, 1, 1, kThreads, true>(c, p, nd, p.n_chunks, mbr);
    if (rc != DSMC_OK) return rc;
    return launch_one<kLmaxBig, kAmaxBig, false, 64, 1, 0, 1, kThreads, true>(c, p, nd, big_grid, mbr);
  }
  if (p.op == 1) {
    // three footprints: 704 slots and 32 cells at 9 CTAs/SM (chunks of cells up to ~230 particles), 1024 slots / 8 cells at 7 CTAs/SM
    // (one ~1000-particle cell), then anything legal on one CTA per SM
    rc = launch_one<704, 32, true, 64, 0, 1, 9, 128>(c, p, nd, p.n_chunks, 0);
    if (rc != DSMC_OK) return rc;
    rc = launch_one<1024, 8, true, 64, 1, 2, 7, 128>(c, p, nd, c->num_sms * 7, 0);
    if (rc != DSMC_OK) return rc;
    return launch_one<kLmaxBig, kAmaxBig, true, 64, 2, 0, 1>(c, p, nd, big_grid, 0);
  }
  nd = *net;
  if (nd.dmax <= 128) {
    const size_t mb = sizeof(float) * 2 * nd.dmax * 64;
    rc = launch_one<kLmaxSmall, kAmaxSmall, false, 64, 0, 1, 1>(c, p, nd, p.n_chunks, mb);
    if (rc != DSMC_OK) return rc;
    return launch_one<kLmaxBig, kAmaxBig, false, 64, 1, 0, 1>(c, p, nd, big_grid, mb);
  }
  const size_t mb = sizeof(float) * 2 * nd.dmax * 32;
  rc = launch_one<kLmaxSmall, kAmaxSmall, false, 32, 0, 1, 1>(c, p, nd, p.n_chunks, mb);
  if (rc != DSMC_OK) return rc;
  return launch_one<kLmaxBig, kAmaxBig, false, 32, 1, 0, 1>(c, p, nd, big_grid, mb);
}

// ---------------------------------------------------------------------------------------------
// a10: chi for independent pairs (BASELINE.json cfg 4)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_chi_batch_table(int64_t n, const float *__restrict__ E,
                                                        const float *__restrict__ b, float *__restrict__ chi,
                                                        ChiTableDev T, float b_scale) {
  for (int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; p < n; p += (int64_t)gridDim.x * blockDim.x)
    chi[p] = chi_table_t(T, table_tE(T, __ldg(E + p)), __ldg(b + p) * b_scale);
}

template <int TP>
__global__ void __launch_bounds__(kThreads) k_chi_batch_mlp(int64_t n, const float *__restrict__ E,
                                                           const float *__restrict__ b, float *__restrict__ chi,
                                                           const MlpDev net, float inv_bmax, float lnE_min,
                                                           float inv_range) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float *buf = reinterpret_cast<float *>(smem_raw);
  const int tid = threadIdx.x;
  const int64_t n_tiles = (n + TP - 1) / TP;
  for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const int64_t p = tile * TP + tid;
    if (tid < TP) {
      float x0 = 0.f, x1 = 0.f;
      if (p < n) {
        float e = (logf(__ldg(E + p)) - lnE_min) * inv_range;
        x0 = !(e > 0.f) ? 0.f : fminf(e, 1.f);
        float bt = __ldg(b + p) * inv_bmax;
        x1 = !(bt > 0.f) ? 0.f : fminf(bt, 1.f);
      }
      buf[tid] = x0;
      buf[TP + tid] = x1;
    }
    __syncthreads();
    const float *out = mlp_tile_fp32<TP>(net, buf);
    if (tid < TP && p < n) {
      const float z = out[tid];
      chi[p] = expm1f(fmaxf(z, 0.f) + log1pf(expf(-fabsf(z))));
    }
    __syncthreads();
  }
}

int launch_chi_batch(dsmc_ctx *c, int64_t n, const float *E, const float *b, float *chi, int mode, float b_max,
                     float lnE_min, float lnE_max, const MlpDev *net) {
  if (mode == 0) {
    const int grid = (int)std::min<int64_t>((n + 255) / 256, (int64_t)c->num_sms * 16);
    k_chi_batch_table<<<grid, 256, 0, c->stream>>>(n, E, b, chi, c->table, (float)(c->table.nB - 1) / b_max);
  } else {
    const MlpDev nd = *net;
    const float inv_range = 1.0f / (lnE_max - lnE_min);
    if (nd.dmax <= 128) {
      const size_t smem = sizeof(float) * 2 * nd.dmax * 64;
      cudaFuncSetAttribute(k_chi_batch_mlp<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      const int grid = (int)std::min<int64_t>((n + 63) / 64, (int64_t)c->num_sms * 2);
      k_chi_batch_mlp<64><<<grid, kThreads, smem, c->stream>>>(n, E, b, chi, nd, 1.0f / b_max, lnE_min, inv_range);
    } else {
      const size_t smem = sizeof(float) * 2 * nd.dmax * 32;
      cudaFuncSetAttribute(k_chi_batch_mlp<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      const int grid = (int)std::min<int64_t>((n + 31) / 32, (int64_t)c->num_sms * 2);
      k_chi_batch_mlp<32><<<grid, kThreads, smem, c->stream>>>(n, E, b, chi, nd, 1.0f / b_max, lnE_min, inv_range);
    }
  }
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? DSMC_OK : DSMC_ERR_CUDA;
}

}  // namespace dsmc
