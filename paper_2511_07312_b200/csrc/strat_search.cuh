// strat_search.cuh - one search step without networks: expansion and policy kernels
// Part of libstrat.so (one translation unit: strat.cu includes these in order).
#pragma once

namespace {
using namespace strat;

// ---- one search step without networks (S3.7)
// Steps 1-2: slot G = r*rollouts + c*L + l of the output environment = root r, opponent
// configuration c (one DETERMINISE stream per configuration), l-th legal action applied (the
// forced first move).  Thread per slot; the root's mask row lives in shared memory.
template <bool kChase>
__global__ void __launch_bounds__(32) k_search_expand(Params Pr, Params Po, int rollouts, uint32_t k0, uint32_t k1,
                                                      const uint32_t* __restrict__ roots, uint32_t* __restrict__ out,
                                                      int* __restrict__ err) {
  __shared__ __align__(16) uint8_t s_state[kStateBytes];
  __shared__ __align__(16) uint32_t s_mask[kBatch * kMaskWords];
  int lane = threadIdx.x, first = blockIdx.x * kBatch;
  int ng = min(kBatch, Po.num_games - first);
  zero_smem16(s_mask, kMaskBytes, lane);
  __syncwarp();
  if (lane < ng) {
    int G = first + lane, r = G / rollouts, s = G - r * rollouts;
    uint32_t W[32];
    const uint4* p = reinterpret_cast<const uint4*>(roots + (size_t)r * kLineWords);
#pragma unroll
    for (int k = 0; k < 8; ++k) { uint4 v = __ldg(p + k); W[4 * k] = v.x; W[4 * k + 1] = v.y; W[4 * k + 2] = v.z; W[4 * k + 3] = v.w; }
    Game root, g;
    unpack_line(W, root);
    const bool keep_log = kChase && Pr.movelog && Po.movelog;  // the copies inherit the root's chase memory
    if (keep_log) copy_game_log(game_log(Pr, (uint32_t)r), game_log(Po, (uint32_t)G));
    uint32_t* row = s_mask + lane * kMaskWords;
    int cnt[4] = {0, 0, 0, 0};
    int L = root.done ? 0 : legal_mask_row(root, root.ply & 1u, rules_of<kChase>(Pr), row, cnt,
                                           kChase ? game_log(Pr, (uint32_t)r) : nullptr);
    int C = L > 0 ? max(1, rollouts / L) : 0;
    int used = min(C * L, rollouts);
    if (s >= used) {  // unused slot: the root, frozen
      g = root; g.done = 1; g.reason = 0; g.result = 0;
      if (!keep_log) g.logn = 0;
    } else {
      int c = s / L, l = s - c * L;
      if (!determinise_game(root, k0, k1, Po.game_base + (uint32_t)(r * rollouts + c), keep_log, g)) raise_error(err, STRAT_BAD_STATE);
      step_game<false, false, kChase>(Po, (uint32_t)G, g, pick_rank(row, cnt, l));
    }
    write_game(s_state, lane, g);
  }
  __syncwarp();
  store_lines(out, first, ng, s_state, lane);
}

// Steps 3-4: per root, qhat(a) = mean over configurations of the value of the game that started
// with a (its result from the searcher's side, 0 while it runs), the magnet policy rho
// and eq. (8).  One CTA per root; float32 arithmetic.  `values` (or null): float32 [R*rollouts] leaf values
// from the searcher's side, used for the games that have not ended (strat_search_policy_values).
constexpr int kPolicyThreads = 128;
template <bool kChase>
__global__ void __launch_bounds__(kPolicyThreads) k_search_policy(Params Pr, int rollouts, const uint32_t* __restrict__ roots,
                                                                  const uint32_t* __restrict__ games,
                                                                  const float* __restrict__ pi_theta,
                                                                  const float* __restrict__ values, float alpha, float beta,
                                                                  float* __restrict__ qhat, float* __restrict__ rho,
                                                                  float* __restrict__ pi_search) {
  __shared__ __align__(16) uint32_t s_row[kMaskWords + 3];
  __shared__ int16_t s_legal[STRAT_NUM_ACTIONS];
  __shared__ int s_q[STRAT_NUM_ACTIONS];      // value sums, then (as float) the logits
  __shared__ int s_cell[100];
  __shared__ int s_L, s_pieces, s_sign;
  __shared__ float s_red[kPolicyThreads / 32];
  const int tid = threadIdx.x, r = blockIdx.x;
  float* q = qhat + (size_t)r * STRAT_NUM_ACTIONS;
  float* rh = rho + (size_t)r * STRAT_NUM_ACTIONS;
  float* ps = pi_search + (size_t)r * STRAT_NUM_ACTIONS;
  for (int a = tid; a < STRAT_NUM_ACTIONS; a += kPolicyThreads) { q[a] = 0.f; rh[a] = 0.f; ps[a] = 0.f; s_q[a] = 0; }
  for (int w = tid; w < kMaskWords + 3; w += kPolicyThreads) s_row[w] = 0;
  if (tid < 100) s_cell[tid] = 0;
  __syncthreads();
  if (tid == 0) {
    uint32_t W[32];
    const uint4* p = reinterpret_cast<const uint4*>(roots + (size_t)r * kLineWords);
#pragma unroll
    for (int k = 0; k < 8; ++k) { uint4 v = __ldg(p + k); W[4 * k] = v.x; W[4 * k + 1] = v.y; W[4 * k + 2] = v.z; W[4 * k + 3] = v.w; }
    Game root;
    unpack_line(W, root);
    int cnt[4] = {0, 0, 0, 0};
    int L = root.done ? 0 : legal_mask_row(root, root.ply & 1u, rules_of<kChase>(Pr), s_row, cnt,
                                           kChase ? game_log(Pr, (uint32_t)r) : nullptr);
    int k = 0, pieces = 0;
    for (int w = 0; w < kMaskWords; ++w)
      for (uint32_t b = s_row[w]; b; b &= b - 1) {
        int a = 32 * w + __ffs((int)b) - 1;
        s_legal[k++] = (int16_t)a;
        if (s_cell[a / 36]++ == 0) ++pieces;
      }
    s_L = L; s_pieces = pieces; s_sign = (root.ply & 1u) ? -1 : 1;
  }
  __syncthreads();
  const int L = s_L;
  if (L == 0) return;
  const int C = max(1, rollouts / L), used = min(C * L, rollouts);
  for (int s = tid; s < used; s += kPolicyThreads) {
    uint32_t f = games[((size_t)r * rollouts + s) * kLineWords + 19] >> 4;
    int v = (f & 1u) ? ((int)((f >> 4) & 3u) - 1) * s_sign : 0;
    if (v) atomicAdd(&s_q[s % L], v);
  }
  __syncthreads();
  // value sums -> float logits in place; a prior without mass on any legal action of this root says
  // nothing here (every logit -inf): the root is then treated as if no prior were given (R29)
  float* logit = reinterpret_cast<float*>(s_q);
  float mx = -INFINITY;
  for (int pass = 0; pass < 2; ++pass) {
    const bool uniform = pi_theta == nullptr || pass == 1;
    mx = -INFINITY;
    for (int l = tid; l < L; l += kPolicyThreads) {
      int a = s_legal[l];
      float qv, rv = 1.0f / ((float)s_pieces * (float)s_cell[a / 36]);
      if (pass == 0) {
        int n = (used - l + L - 1) / L;  // games that started with this action
        qv = n ? (float)s_q[l] / (float)n : 0.f;
        if (values) {
          // caller-supplied leaf values for the games still running, the result for the finished
          // ones; summed per action in slot order in double, so that qhat is the same number on every run
          double sum = 0.0;
          for (int s = l; s < used; s += L) {
            const uint32_t f = games[((size_t)r * rollouts + s) * kLineWords + 19] >> 4;
            sum += (f & 1u) ? (double)(((int)((f >> 4) & 3u) - 1) * s_sign) : (double)values[(size_t)r * rollouts + s];
          }
          qv = n ? (float)(sum / (double)n) : 0.f;
        }
        q[a] = qv; rh[a] = rv;
      } else {
        qv = q[a];
      }
      float pv = uniform ? 1.0f / (float)L : pi_theta[(size_t)r * STRAT_NUM_ACTIONS + a];
      float lg = (qv + alpha * logf(rv) + beta * logf(pv)) / (alpha + beta);
      logit[l] = lg;
      mx = fmaxf(mx, lg);
    }
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, off));
    if ((tid & 31) == 0) s_red[tid >> 5] = mx;
    __syncthreads();
    mx = fmaxf(fmaxf(s_red[0], s_red[1]), fmaxf(s_red[2], s_red[3]));
    __syncthreads();
    if (mx > -INFINITY || uniform) break;  // the same decision in every thread
  }
  float z = 0.f;
  for (int l = tid; l < L; l += kPolicyThreads) { float e = expf(logit[l] - mx); logit[l] = e; z += e; }
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) z += __shfl_xor_sync(0xffffffffu, z, off);
  if ((tid & 31) == 0) s_red[tid >> 5] = z;
  __syncthreads();
  z = (s_red[0] + s_red[1]) + (s_red[2] + s_red[3]);
  for (int l = tid; l < L; l += kPolicyThreads) ps[s_legal[l]] = logit[l] / z;
}


}  // namespace
