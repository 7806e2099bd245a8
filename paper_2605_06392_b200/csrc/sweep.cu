// Host orchestration of the sweeps over the nt time blocks (sequential in t, parallel inside each block).
//   forward : Algorithm 1 (R8) -- blocked POTRF + TRTRI of D_t - S_{t-1}, L_B = B X^T,
//             Schur update of D_{t+1}, arrow rows and right-hand-side rows, tip.
//   backward: Eqs. 3-5 + BTA selected inversion (R10) + the Eq. 7
//             trace contractions fused per block (only Z_Dt and Z_D{t+1} are live).
// The factor is held in inverse-diagonal form X_t = L_Dt^-1, so every large step is a GEMM (gemm.cu).
#include <cstdlib>

#include "sweep.h"

#define CK(call)                      \
  do {                                \
    cudaError_t e_ = (call);          \
    if (e_ != cudaSuccess) return e_; \
  } while (0)

// Two lanes per chain: its normal stream for the full-chip kernels and (optionally) a high-priority companion stream
// for the small latency-bound ones (POTRF leaves, small GEMMs of the recursion, skinny / tip / contraction kernels).
// The block scheduler serves pending CTAs of higher-priority streams first, so a one-CTA leaf of this chain is not
// queued behind the hundreds of pending CTAs of another chain's GEMM.  Switching lanes costs one event.
cudaStream_t lane(Chain* ch, cudaStream_t big, bool small) {
  if (!ch || !ch->hi) return big;
  if (ch->on_small != small) {
    bta_ctx* c = ch->c;
    cudaEvent_t e = c->ev_sw[(c->ev_sw_next++) % BTA_NSW];
    cudaStream_t from = ch->on_small ? ch->hi : big, to = small ? ch->hi : big;
    cudaEventRecord(e, from);
    cudaStreamWaitEvent(to, e, 0);
    ch->on_small = small;
  }
  return small ? ch->hi : big;
}
cudaError_t chain_to_big(Chain& ch, cudaStream_t big) {
  lane(&ch, big, false);
  if (ch.rows_pending && ch.rs && ch.rs != big) {  // fold the rows stream in as well
    cudaEvent_t e = ch.c->ev_sw[(ch.c->ev_sw_next++) % BTA_NSW];
    cudaEventRecord(e, ch.rs);
    cudaStreamWaitEvent(big, e, 0);
  }
  ch.rows_pending = false;
  if (ch.solve_pending && ch.ss && ch.ss != big) {  // ... and the solve stream
    cudaEvent_t e = ch.c->ev_sw[(ch.c->ev_sw_next++) % BTA_NSW];
    cudaEventRecord(e, ch.ss);
    cudaStreamWaitEvent(big, e, 0);
  }
  ch.solve_pending = false;
  if (ch.g_pending && ch.gs && ch.gs != big) {
    cudaEvent_t e = ch.c->ev_sw[(ch.c->ev_sw_next++) % BTA_NSW];
    cudaEventRecord(e, ch.gs);
    cudaStreamWaitEvent(big, e, 0);
  }
  ch.g_pending = false;
  return cudaGetLastError();
}
#define SS lane(lch, st, true)
#define SB lane(lch, st, false)

namespace {
inline GemmArgs G(int mode, int M, int N, int K, double alpha, const double* A, int lda, const double* B, int ldb,
                  double beta, double* C, int ldc, int klo, int khi, int out) {
  return GemmArgs{A, B, C, M, N, K, lda, ldb, ldc, alpha, beta, mode, klo, khi, out, nullptr, 0, 0};
}
}  // namespace

namespace {
// a GEMM of the recursion goes to the small lane when it runs with the small-tile configuration
cudaError_t gemm_lane(Chain* lch, cudaStream_t st, const GemmArgs& g) {
  return launch_gemm(g, gemm_uses_small_tiles(g) ? SS : SB);
}
}  // namespace

// A[lo:hi, lo:hi] (lower, SPD) -> X = L^-1 in place; T1, T2: scratch with the same leading dimension.
// Recursive on 128-wide tiles (leaf: leaf.cu):  chol/inv(A11);  L21 = A21 X11^T;  A22 -= L21 L21^T;  chol/inv(A22);
// X21 = -X22 (L21 X11).  b^3/3 (POTRF) + b^3/3 (TRTRI) flops, all but the 128x128 leaves in DMMA GEMMs.
// Recursive on 128-wide tiles; a remainder of up to 16 rows stays with the last tile (the leaf takes 144 rows).
constexpr int TILE = 128;
int potrf_split(int n) {
  if (n <= leaf_max_n()) return n;
  const int ntile = (n - (leaf_max_n() - TILE) + TILE - 1) / TILE;
  return TILE * ((ntile + 1) / 2);
}

cudaError_t potrf_inv(bta_ctx* c, Chain* lch, double* A, int ld, int lo, int hi, double* T1, double* T2, double* diagL,
                      long long grow0, cudaStream_t st, int phase) {
  const int n = hi - lo;
  if (n <= 0) return cudaSuccess;
  if (n <= leaf_max_n()) {
    if (phase == 2) return cudaSuccess;
    BTA_COUNT(c);
    return launch_potrf_inv_blocked(A + (long long)lo * ld + lo, ld, n, diagL ? diagL + lo : nullptr, grow0 + lo,
                                 c->pivot_flag, SS);
  }
  const int mid = lo + potrf_split(n);
  const int s1 = mid - lo, s2 = hi - mid;
  const bool top = lch && n == ld && c->trace_on;
#define PM(tag) \
  if (top) trace_mark(c, lane(lch, st, lch->on_small), lch->trace_id, (int)(grow0 / ld), tag)
  if (phase != 2) CK(potrf_inv(c, lch, A, ld, lo, mid, T1, T2, diagL, grow0, st));
  if (phase == 1) return cudaSuccess;
  PM(10);
  double* A11 = A + (long long)lo * ld + lo;
  double* A21 = A + (long long)mid * ld + lo;
  double* A22 = A + (long long)mid * ld + mid;
  double* L21 = T1 + (long long)mid * ld + lo;
  double* LX = T2 + (long long)mid * ld + lo;
  CK(gemm_lane(lch, st, G(GEMM_NT, s2, s1, s1, 1.0, A21, ld, A11, ld, 0.0, L21, ld, KLO_ZERO, KHI_NEND, OUT_FULL)));
  // L21 X11 feeds only X21 at the end of this level.  Where a step is latency-bound (b <= 1024: the chip is not full) it
  // runs on the chain's side stream beside the update and the factorisation of A22 instead of after them.  (Above that
  // size the same move costs 3-11 %: DESIGN.md §6.)
  const bool lx_side = lch && lch->xs && ld <= 1024 && n < ld;
  cudaEvent_t e_lx = nullptr;
  if (lx_side) {
    cudaEvent_t e0 = c->ev_sw[(c->ev_sw_next++) % BTA_NSW];
    e_lx = c->ev_sw[(c->ev_sw_next++) % BTA_NSW];
    CK(cudaEventRecord(e0, lane(lch, st, lch->on_small)));   // L21 (and X11) are complete in lane order
    CK(cudaStreamWaitEvent(lch->xs, e0, 0));
    CK(launch_gemm(G(GEMM_NN, s2, s1, s1, 1.0, L21, ld, A11, ld, 0.0, LX, ld, KLO_N0, KHI_K, OUT_FULL), lch->xs));
    CK(cudaEventRecord(e_lx, lch->xs));
  }
  CK(gemm_lane(lch, st, G(GEMM_NT, s2, s2, s1, -1.0, L21, ld, L21, ld, 1.0, A22, ld, KLO_ZERO, KHI_K, OUT_LOWER)));
  c->launches += 2;
  PM(11);
  CK(potrf_inv(c, lch, A, ld, mid, hi, T1, T2, diagL, grow0, st));
  PM(12);
  if (lx_side) {
    const GemmArgs gx = G(GEMM_NN, s2, s1, s2, -1.0, A22, ld, LX, ld, 0.0, A21, ld, KLO_ZERO, KHI_MEND, OUT_FULL);
    cudaStream_t tgt = gemm_uses_small_tiles(gx) ? SS : SB;
    CK(cudaStreamWaitEvent(tgt, e_lx, 0));
    CK(launch_gemm(gx, tgt));
  } else {
    CK(gemm_lane(lch, st, G(GEMM_NN, s2, s1, s1, 1.0, L21, ld, A11, ld, 0.0, LX, ld, KLO_N0, KHI_K, OUT_FULL)));
    CK(gemm_lane(lch, st, G(GEMM_NN, s2, s1, s2, -1.0, A22, ld, LX, ld, 0.0, A21, ld, KLO_ZERO, KHI_MEND, OUT_FULL)));
  }
  c->launches += 2;
  return cudaSuccess;
}

// Forward step with the coupling block folded into the top level of the POTRF+TRTRI recursion (factor mode).
// With A = [[A11, .], [A21, A22]], X = L^-1 = [[X11, 0], [X21, X22]] and B = [B1 | B2]:
//   L_B = B X^T = [ B1 X11^T | (B2 - L_B1 L21^T) X22^T ],   S = L_B1 L_B1^T + L_B2 L_B2^T,   X21 = -X22 (L21 X11).
// L_B1, B2 - L_B1 L21^T and L_B1's half of the Schur update need only X11 (and L21), and X21 is not needed by the
// factorisation at all, so they run on the chain's side stream `xs` next to the second half of the recursion; the
// dependent chain of a step is potrf_inv(A11) -> L21, A22 -> potrf_inv(A22) -> (.) X22^T -> second half of S instead
// of ... -> X21 -> L_B -> S.  Same
// flops.  B (its right half) is updated in place; L_B goes to `dst`.
cudaError_t potrf_inv_coupled(bta_ctx* c, Chain* lch, double* A, int b, double* Bi, double* dst, double* Dnext,
                              double* T1, double* T2, double* diagL, long long grow0, cudaStream_t st,
                              cudaStream_t xs) {
  Chain& ch = *lch;
  const int t = (int)(grow0 / b);
  const int mid = potrf_split(b);
  const int s1 = mid, s2 = b - mid, ld = b;
  auto ev_next = [&]() { return c->ev_sw[(c->ev_sw_next++) % BTA_NSW]; };
  auto cur = [&]() { return lane(lch, st, ch.on_small); };
#define XM(tag) trace_mark(c, cur(), ch.trace_id, t, tag)
  CK(potrf_inv(c, lch, A, ld, 0, mid, T1, T2, diagL, grow0, st));
  XM(10);
  cudaEvent_t e1 = ev_next(), e2 = ev_next(), e3 = ev_next(), e4 = ev_next(), e5 = ev_next();
  CK(cudaEventRecord(e1, cur()));
  CK(cudaStreamWaitEvent(xs, e1, 0));
  //   side: L_B1 = B1 X11^T, S += L_B1 L_B1^T
  CK(launch_gemm(G(GEMM_NT, b, s1, s1, 1.0, Bi, b, A, ld, 0.0, dst, b, KLO_ZERO, KHI_NEND, OUT_FULL), xs));
  CK(cudaEventRecord(e2, xs));
  //   main: second half of the recursion
  double* A21 = A + (long long)mid * ld;
  double* A22 = A + (long long)mid * ld + mid;
  double* L21 = T1 + (long long)mid * ld;
  double* LX = T2 + (long long)mid * ld;
  CK(gemm_lane(lch, st, G(GEMM_NT, s2, s1, s1, 1.0, A21, ld, A, ld, 0.0, L21, ld, KLO_ZERO, KHI_NEND, OUT_FULL)));
  cudaEvent_t e6 = ev_next(), e7 = ev_next();
  CK(cudaEventRecord(e6, cur()));
  CK(gemm_lane(lch, st, G(GEMM_NT, s2, s2, s1, -1.0, L21, ld, L21, ld, 1.0, A22, ld, KLO_ZERO, KHI_K, OUT_LOWER)));
  c->launches += 2;
  //   side: B2 -= L_B1 L21^T (needs only L_B1 and L21: beside the factorisation of A22), then S += L_B1 L_B1^T
  CK(cudaStreamWaitEvent(xs, e6, 0));
  CK(launch_gemm(G(GEMM_NT, b, s2, s1, -1.0, dst, b, L21, ld, 1.0, Bi + mid, b, KLO_ZERO, KHI_K, OUT_FULL), xs));
  CK(cudaEventRecord(e7, xs));
  if (Dnext)
    CK(launch_gemm(G(GEMM_NT, b, b, s1, -1.0, dst, b, dst, b, 1.0, Dnext, b, KLO_ZERO, KHI_K, OUT_LOWER), xs));
  CK(cudaEventRecord(e3, xs));
  c->launches += Dnext ? 3 : 2;
  XM(11);
  CK(potrf_inv(c, lch, A, ld, mid, b, T1, T2, diagL, grow0, st));
  XM(12);
  //   side: X21 = -X22 (L21 X11), off the dependent chain
  CK(cudaEventRecord(e4, cur()));
  CK(cudaStreamWaitEvent(xs, e4, 0));
  CK(launch_gemm(G(GEMM_NN, s2, s1, s1, 1.0, L21, ld, A, ld, 0.0, LX, ld, KLO_N0, KHI_K, OUT_FULL), xs));
  CK(launch_gemm(G(GEMM_NN, s2, s1, s2, -1.0, A22, ld, LX, ld, 0.0, A21, ld, KLO_ZERO, KHI_MEND, OUT_FULL), xs));
  CK(cudaEventRecord(e5, xs));
  c->launches += 2;
  //   main: L_B2 = (B2 - L_B1 L21^T) X22^T, S += L_B2 L_B2^T
  CK(cudaStreamWaitEvent(SB, e7, 0));
  CK(launch_gemm(G(GEMM_NT, b, s2, s2, 1.0, Bi + mid, b, A22, ld, 0.0, dst + mid, b, KLO_ZERO, KHI_NEND, OUT_FULL),
                 SB));
  c->launches += 1;
  XM(3);
  CK(cudaStreamWaitEvent(SB, e3, 0));
  if (Dnext) {
    CK(launch_gemm(G(GEMM_NT, b, b, s2, -1.0, dst + mid, b, dst + mid, b, 1.0, Dnext, b, KLO_ZERO, KHI_K, OUT_LOWER),
                   SB));
    BTA_COUNT(c);
  }
  CK(cudaStreamWaitEvent(SB, e5, 0));
  XM(4);
#undef XM
  return cudaSuccess;
}

namespace {
__global__ void tip_init_kernel(int a, int nr, const double* __restrict__ T, int ldt_in,
                                const double* __restrict__ rhs_tip, int tip_stride, double* __restrict__ Tt, int zero) {
  const int p = threadIdx.x / (a + nr), q = threadIdx.x % (a + nr);
  if (p >= a) return;
  double v = 0.0;
  if (!zero) v = (q < a) ? T[p * ldt_in + q] : rhs_tip[(long long)(q - a) * tip_stride + p];
  Tt[p * (a + nr) + q] = v;
}
__global__ void tip_add_kernel(int n, const double* __restrict__ src, double* __restrict__ dst) {
  if (threadIdx.x < n) dst[threadIdx.x] += src[threadIdx.x];
}
__global__ void scale_copy_kernel(long long n, double alpha, const double* __restrict__ in, double* __restrict__ out) {
  long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e < n) out[e] = alpha * in[e];
}
}  // namespace

cudaError_t chain_forward_begin(Chain& ch, cudaStream_t st) {
  Chain* lch = &ch;
  bta_ctx* c = ch.c;
  const int a = ch.a, ldt = a + ch.nr;
  if (a > 0) {
    tip_init_kernel<<<1, a * ldt, 0, SS>>>(a, ch.nr, ch.T, ch.ldT, ch.rhs_tip, ch.rhs_tip_stride, ch.Tt,
                                           ch.tt_zero ? 1 : 0);
    BTA_COUNT(c);
  }
  return cudaGetLastError();
}

cudaError_t chain_forward_step(Chain& ch, int t, cudaStream_t st) {
  Chain* lch = &ch;
  bta_ctx* c = ch.c;
  const int b = ch.b, nt = ch.nt, a = ch.a, P = ch.P(), ldt = a + ch.nr;
  const long long bb = (long long)b * b;
  const long long tg = ch.tg(t);                  // global time block (diag(L) position, pivot row)
  double* At = ch.Dp(t);           // D_t - S_{t-1}
  double* Dt = ch.carry ? ch.Xs : At;            // where X_t = L_Dt^-1 is built
  const double* LBprev = ch.carry ? ch.LBs : (t > 0 ? ch.Bout + (t - 1) * ch.b_stride : nullptr);
  // Forward pipelining: when the previous step issued its products in split form (see the end of this function), the
  // first half of this block's POTRF+TRTRI (A11 = the top-left part of D_t - S_{t-1}) depends only on the first two of
  // those five launches.  It starts now on the chain's priority lane, next to the rest of the previous step's products
  // on the main lane -- the chain offers the GPU latency-bound and chip-filling work at the same time.
  constexpr int split_maxb = 1024;  // the coupled step (below) pays only where a step is latency-bound
  const bool can_pipe = ch.pipe_ev && ch.hi && c->opt.pipeline && ch.factor_blocks && !ch.carry && !ch.zero_upper &&
                        b > split_maxb;
  bool early = false;
  if (can_pipe && ch.pipe_armed) {
    ch.on_small = true;  // enter the priority lane WITHOUT ordering it after the tail of the main lane ...
    CK(cudaStreamWaitEvent(ch.hi, ch.pipe_ev[0], 0));  // ... only after the Schur update of A11
    CK(potrf_inv(c, lch, At, b, 0, b, ch.W2, ch.W3, ch.dvec ? ch.dvec + tg * b : nullptr, tg * b, st, 1));
    early = true;
  }
  // stack rows: arrow rows (factor mode) then right-hand-side rows.
  //   R~_t = R_t - R^_{t-1} L_B{t-1}^T  (lines 4-5), done first: in carry mode L_B{t-1} is overwritten below
  // Factor mode with a rows stream: all row work of this step is issued at its end on that stream (see there).
  const bool defer_rows = ch.rs && P > 0 && ch.factor_blocks && !ch.carry && !ch.Rtmp && ch.Rin != ch.Rout &&
                          !ch.arrow_given;
  const double* src = nullptr;
  int ld_src = 0;
  if (P > 0 && !defer_rows) {
    src = ch.Rin + t * ch.rin_stride;
    ld_src = ch.ld_rin;
    if (t == 0 && ch.Rin == ch.Rout) {  // in-place factor: the stack product below must not alias its input
      CK(cudaMemcpy2DAsync(ch.Rtmp, b * sizeof(double), src, ld_src * sizeof(double), b * sizeof(double), P,
                           cudaMemcpyDeviceToDevice, SS));
      src = ch.Rtmp;
      ld_src = b;
    }
    if (t > 0) {
      if (early) CK(cudaStreamWaitEvent(SS, ch.pipe_ev[1], 0));  // L_B{t-1} is complete
      double* tmp = ch.Rtmp ? ch.Rtmp : ch.Rin + t * ch.rin_stride;
      const int ld_tmp = ch.Rtmp ? b : ch.ld_rin;
      CK(launch_skinny_nt(P, b, b, ch.Rout + (t - 1) * ch.rout_stride, ch.ld_rout, LBprev, b, 0, -1.0, 1.0, src, ld_src,
                          tmp, ld_tmp, SS));
      BTA_COUNT(c);
      src = tmp;
      ld_src = ld_tmp;
    }
  }
  if (early)  // everything else of this step comes after all products of the previous step
    CK(cudaStreamWaitEvent(lane(lch, st, ch.on_small), ch.pipe_ev[2], 0));
  ch.pipe_armed = false;
#define TM(tag) trace_mark(c, lane(lch, st, ch.on_small), ch.trace_id, t, tag)
  TM(0);
  bool coupled = false;  // L_B and the Schur update were folded into the recursion (potrf_inv_coupled)
  if (ch.factor_blocks) {
    if (ch.zero_upper) {
      CK(launch_zero_upper(At, b, b, SB));
      BTA_COUNT(c);
    }
    if (ch.carry) {  // the carry D_t - S_{t-1} stays in its slot; factor a copy
      CK(cudaMemcpyAsync(Dt, At, bb * sizeof(double), cudaMemcpyDeviceToDevice, SB));
      if (ch.ring) {  // host staging: the carry is final (S_{t-1} was applied in main-lane order) -- copy it out
        cudaEvent_t e = c->ev_sw[(c->ev_sw_next++) % BTA_NSW];
        CK(cudaEventRecord(e, SB));
        CK(cudaStreamWaitEvent(ch.cs, e, 0));
        CK(cudaMemcpyAsync(ch.hostD + (long long)t * bb, At, bb * sizeof(double), cudaMemcpyDeviceToHost, ch.cs));
        CK(cudaEventRecord(ch.ring_ev[t % ch.ring], ch.cs));
      }
      CK(potrf_inv(c, lch, Dt, b, 0, b, ch.W1, ch.Bs, ch.dvec ? ch.dvec + tg * b : nullptr, tg * b, st));
    } else {
      const bool has_coupling = t < nt - 1 || ch.tail_coupling;
      coupled = has_coupling && ch.xs && b > leaf_max_n() && b <= split_maxb;
      if (coupled) {
        double* Bi = ch.Bin + t * ch.b_stride;
        double* Bo = ch.Bout + t * ch.b_stride;
        double* dst = (Bi == Bo) ? ch.W1 : Bo;
        CK(potrf_inv_coupled(c, lch, Dt, b, Bi, dst, t < nt - 1 ? ch.Dp(t + 1) : nullptr, ch.W2, ch.W3,
                             ch.dvec ? ch.dvec + tg * b : nullptr, tg * b, st, ch.xs));
        if (dst != Bo) CK(cudaMemcpyAsync(Bo, dst, bb * sizeof(double), cudaMemcpyDeviceToDevice, SB));
      } else {
        CK(potrf_inv(c, lch, Dt, b, 0, b, ch.W2, ch.W3, ch.dvec ? ch.dvec + tg * b : nullptr, tg * b, st, early ? 2 : 0));
      }
    }
  }
  TM(1);
  if (P > 0 && !defer_rows) {
    //   R^_t = R~_t X_t^T
    double* Rh = ch.Rout + t * ch.rout_stride;
    CK(launch_skinny_nt(P, b, b, src, ld_src, Dt, b, 1, 1.0, 0.0, nullptr, 0, Rh, ch.ld_rout, SS));
    BTA_COUNT(c);
    if (a > 0) {
      // T~ -= L_C L_C^T (line 9) and r_T - v_T, v_T += L_C z (line 5): columns [0,a) and [a, a+nr) of Tt
      if (ch.arrow_rows) {
        CK(launch_small_nt(a, P, b, Rh, ch.ld_rout, Rh, ch.ld_rout, -1.0, ch.Tt, ldt, SS));
        BTA_COUNT(c);
      } else if (ch.arrow_given) {
        CK(launch_small_nt(a, ch.nr, b, ch.LCgiven + t * ch.lc_stride, b, Rh, ch.ld_rout, -1.0, ch.Tt + a, ldt, SS));
        BTA_COUNT(c);
      }
    }
  }
  if ((t < nt - 1 || ch.tail_coupling) && ch.factor_blocks && !coupled) {
    const double* Bi;
    double *Bo, *dst;
    if (ch.carry) {
      CK(launch_assemble_block(c, ch.which, 1, ch.tB(t), ch.transposeB ? 1 : 0, ch.Bs, SB));
      Bi = ch.Bs;
      Bo = dst = ch.LBs;
    } else {
      Bi = ch.Bin + t * ch.b_stride;
      Bo = ch.Bout + t * ch.b_stride;
      dst = (Bi == Bo) ? ch.W1 : Bo;
    }
    TM(2);
    if (can_pipe && t < nt - 1) {
      // Split form: rows [0, h) of L_B and the top-left h x h part of the Schur update first (h = the next block's
      // A11), then the rest.  Same flops.
      double* Dn = ch.Dp(t + 1);
      const int h = potrf_split(b), r = b - h;
      const long long ho = (long long)h * b;
      CK(launch_gemm(G(GEMM_NT, h, b, b, 1.0, Bi, b, Dt, b, 0.0, dst, b, KLO_ZERO, KHI_NEND, OUT_FULL), SB));
      CK(launch_gemm(G(GEMM_NT, h, h, b, -1.0, dst, b, dst, b, 1.0, Dn, b, KLO_ZERO, KHI_K, OUT_LOWER), SB));
      CK(cudaEventRecord(ch.pipe_ev[0], SB));
      CK(launch_gemm(G(GEMM_NT, r, b, b, 1.0, Bi + ho, b, Dt, b, 0.0, dst + ho, b, KLO_ZERO, KHI_NEND, OUT_FULL), SB));
      CK(cudaEventRecord(ch.pipe_ev[1], SB));
      TM(3);
      CK(launch_gemm(G(GEMM_NT, r, h, b, -1.0, dst + ho, b, dst, b, 1.0, Dn + ho, b, KLO_ZERO, KHI_K, OUT_FULL), SB));
      CK(launch_gemm(G(GEMM_NT, r, r, b, -1.0, dst + ho, b, dst + ho, b, 1.0, Dn + ho + h, b, KLO_ZERO, KHI_K,
                       OUT_LOWER),
                     SB));
      c->launches += 5;
      if (dst != Bo) CK(cudaMemcpyAsync(Bo, dst, bb * sizeof(double), cudaMemcpyDeviceToDevice, SB));
      CK(cudaEventRecord(ch.pipe_ev[2], SB));
      ch.pipe_armed = true;
    } else {
      CK(launch_gemm(G(GEMM_NT, b, b, b, 1.0, Bi, b, Dt, b, 0.0, dst, b, KLO_ZERO, KHI_NEND, OUT_FULL), SB));
      BTA_COUNT(c);
      TM(3);
      if (t < nt - 1) {  // the Schur update of a separator is applied by the separator stage (two chains meet there)
        CK(launch_gemm(G(GEMM_NT, b, b, b, -1.0, dst, b, dst, b, 1.0, ch.Dp(t + 1), b, KLO_ZERO, KHI_K,
                         OUT_LOWER),
                       SB));
        BTA_COUNT(c);
      }
      if (dst != Bo) CK(cudaMemcpyAsync(Bo, dst, bb * sizeof(double), cudaMemcpyDeviceToDevice, SB));
    }
    TM(4);
  }
  if (ch.fill) {  // middle partition: the fill coupling to the top boundary block (sweep.h: Fill)
    Fill& f = *ch.fill;
    double* LF = f.LF + t * f.lf_stride;
    const double* LB = ch.Bout + t * ch.b_stride;
    CK(launch_gemm(G(GEMM_NT, b, b, b, 1.0, f.Ftil, b, Dt, b, 0.0, LF, b, KLO_ZERO, KHI_NEND, OUT_FULL), SB));
    CK(launch_gemm(G(GEMM_NT, b, b, b, -1.0, LF, b, LF, b, 1.0, f.Ds, b, KLO_ZERO, KHI_K, OUT_LOWER), SB));
    if (t < nt - 1)
      CK(launch_gemm(G(GEMM_NT, b, b, b, -1.0, LF, b, LB, b, 0.0, f.Ftil, b, KLO_ZERO, KHI_K, OUT_FULL), SB));
    else
      CK(launch_gemm(G(GEMM_NT, b, b, b, -1.0, LB, b, LF, b, 0.0, f.Bse, b, KLO_ZERO, KHI_K, OUT_FULL), SB));
    c->launches += 3;
    if (P > 0 && !defer_rows) {
      CK(launch_skinny_nt(P, b, b, ch.Rout + t * ch.rout_stride, ch.ld_rout, LF, b, 0, -1.0, 1.0, f.Rs, f.ld_rs, f.Rs,
                          f.ld_rs, SS));
      BTA_COUNT(c);
    }
  }
  if (defer_rows) {
    // everything this step produced (X_t, L_Bt, L_Ft) is complete in the order of the chain's current lane
    cudaStream_t cur = lane(lch, st, ch.on_small), rs = ch.rs;
    cudaEvent_t e = c->ev_sw[(c->ev_sw_next++) % BTA_NSW];
    CK(cudaEventRecord(e, cur));
    CK(cudaStreamWaitEvent(rs, e, 0));
    double* Rt = ch.Rin + t * ch.rin_stride;
    double* Rh = ch.Rout + t * ch.rout_stride;
    if (t > 0) {
      CK(launch_skinny_nt(P, b, b, ch.Rout + (t - 1) * ch.rout_stride, ch.ld_rout, ch.Bout + (t - 1) * ch.b_stride, b, 0,
                          -1.0, 1.0, Rt, ch.ld_rin, Rt, ch.ld_rin, rs));
      BTA_COUNT(c);
    }
    CK(launch_skinny_nt(P, b, b, Rt, ch.ld_rin, Dt, b, 1, 1.0, 0.0, nullptr, 0, Rh, ch.ld_rout, rs));
    BTA_COUNT(c);
    if (a > 0 && ch.arrow_rows) {
      CK(launch_small_nt(a, P, b, Rh, ch.ld_rout, Rh, ch.ld_rout, -1.0, ch.Tt, ldt, rs));
      BTA_COUNT(c);
    }
    if (ch.fill) {
      Fill& f = *ch.fill;
      CK(launch_skinny_nt(P, b, b, Rh, ch.ld_rout, f.LF + t * f.lf_stride, b, 0, -1.0, 1.0, f.Rs, f.ld_rs, f.Rs, f.ld_rs,
                          rs));
      BTA_COUNT(c);
    }
    ch.rows_pending = true;
  }
  return cudaSuccess;
}

cudaError_t chain_forward_end(Chain& ch, cudaStream_t st) {
  Chain* lch = &ch;
  bta_ctx* c = ch.c;
  if (ch.rows_pending) CK(chain_to_big(ch, st));  // the tip accumulator is complete
  const int b = ch.b, nt = c->md.nt, a = ch.a;  // the tip sits after all nt blocks, whatever this chain's length
  if (a > 0) {
    CK(launch_tip(ch.Tt, a, ch.nr, ch.tip_chol ? 1 : 0, ch.LT, ch.zT, ch.xT, ch.ZT,
                  ch.dvec ? ch.dvec + (long long)nt * b : nullptr, (long long)nt * b, c->pivot_flag, SS));
    BTA_COUNT(c);
  }
  return cudaSuccess;
}

// Two-way elimination: the up chain (blocks 0..h-1) and the down chain (blocks nt-1..h+1, time-reversed, with
// transposed coupling blocks) have been eliminated independently; both couple to the separator block h through
// their last L_B.  Apply their Schur updates, arrow/rhs updates and tip contributions to the separator chain `cs`
// (one block, its Rin rows and D already assembled), which is then factored like a last block.
cudaError_t separator_merge_forward(Chain& up, Chain& dn, Chain& cs, cudaStream_t st) {
  Chain* lch = &cs;
  bta_ctx* c = cs.c;
  const int b = cs.b, a = cs.a, P = cs.P();
  Chain* sub[2] = {&up, &dn};
  if (a > 0) {
    tip_add_kernel<<<1, 32 * ((a * (a + cs.nr) + 31) / 32), 0, SS>>>(a * (a + cs.nr), dn.Tt, up.Tt);
    BTA_COUNT(c);
  }
  for (Chain* q : sub) {
    const int last = q->nt - 1;
    const double* LB = q->carry ? q->LBs : q->Bout + last * q->b_stride;
    if (P > 0) {
      CK(launch_skinny_nt(P, b, b, q->Rout + last * q->rout_stride, q->ld_rout, LB, b, 0, -1.0, 1.0, cs.Rin, cs.ld_rin,
                          cs.Rin, cs.ld_rin, SS));
      BTA_COUNT(c);
    }
    CK(launch_gemm(G(GEMM_NT, b, b, b, -1.0, LB, b, LB, b, 1.0, cs.D, b, KLO_ZERO, KHI_K, OUT_LOWER), SB));
    BTA_COUNT(c);
  }
  return cudaSuccess;
}

cudaError_t chain_forward(Chain& ch, cudaStream_t st) {
  CK(chain_forward_begin(ch, st));
  for (int t = 0; t < ch.nt; ++t) CK(chain_forward_step(ch, t, st));
  return chain_forward_end(ch, st);
}

// Backward sweep t = nt-1 .. 0.  Needs from the forward sweep: X_t in D(t), L_Bt in Bout(t), the arrow factor
// rows L_Ct, z_t (rows a.. of Rout(t) when arrow_rows, else rows 0..), and the tip outputs x_T, Z_T.
cudaError_t chain_backward_step(Chain& ch, int t, cudaStream_t st) {
  Chain* lch = ch.lanes_bwd ? &ch : nullptr;
  bta_ctx* c = ch.c;
  const int b = ch.b, nt = ch.nt, a = ch.a, nr = ch.nr;
  const long long bb = (long long)b * b;
  const bool arrow = ch.arrow();
  const int zrow0 = ch.arrow_rows ? a : 0;  // first rhs row inside the Rout stack
  const bool has_next = (t < nt - 1) || ch.tail_coupling;   // a block eliminated after this one couples to it
  const long long tg = ch.tg(t);
  {
    if (ch.carry) {
      // carry-based reconstruction: X_t from the stored D_t - S_{t-1}, L_Bt from the re-assembled B_t
      if (ch.ring) CK(cudaStreamWaitEvent(SB, ch.ring_ev[t % ch.ring], 0));  // the carry is back in its slot
      CK(cudaMemcpyAsync(ch.Xs, ch.Dp(t), bb * sizeof(double), cudaMemcpyDeviceToDevice, SB));
      if (ch.ring && t - ch.ring >= 0) {  // the slot is free: stream block t - ring back from the host
        cudaEvent_t e = c->ev_sw[(c->ev_sw_next++) % BTA_NSW];
        CK(cudaEventRecord(e, SB));
        CK(cudaStreamWaitEvent(ch.cs, e, 0));
        CK(cudaMemcpyAsync(ch.Dp(t), ch.hostD + (long long)(t - ch.ring) * bb, bb * sizeof(double),
                           cudaMemcpyHostToDevice, ch.cs));
        CK(cudaEventRecord(ch.ring_ev[t % ch.ring], ch.cs));
      }
      CK(potrf_inv(c, lch, ch.Xs, b, 0, b, ch.W1, ch.Bs, nullptr, (long long)ch.tg(t) * b, st));
      if (has_next) {
        CK(launch_assemble_block(c, ch.which, 1, ch.tB(t), ch.transposeB ? 1 : 0, ch.Bs, SB));
        CK(launch_gemm(G(GEMM_NT, b, b, b, 1.0, ch.Bs, b, ch.Xs, b, 0.0, ch.LBs, b, KLO_ZERO, KHI_NEND, OUT_FULL), SB));
        BTA_COUNT(c);
      }
    }
    const double* X = ch.carry ? ch.Xs : ch.Dp(t);
    double* LB = has_next ? (ch.carry ? ch.LBs : ch.Bout + t * ch.b_stride) : nullptr;
    const double* LC = nullptr;
    int ld_lc = b;
    if (ch.arrow_rows) {
      LC = ch.Rout + t * ch.rout_stride;
      ld_lc = ch.ld_rout;
    } else if (ch.arrow_given) {
      LC = ch.LCgiven + t * ch.lc_stride;
    }
    // ---- upper solve (Eqs. 3-5):  u = z_t - L_Bt^T x_{t+1} - L_Ct^T x_T ;  x_t = X_t^T u  (row-vector form)
    const bool use_ss = ch.ss && ch.selinv && !ch.selinv_inplace && !ch.carry && !ch.fill;
    const bool side_solve = nr > 0 && use_ss && ch.part2;
    const bool side_g = use_ss && ch.gs && has_next && ch.pipe_ev && ch.Gm2[t & 1];
    cudaEvent_t ev_solve = nullptr;   // the work of this step on the solve stream has read L_Bt
    if ((side_solve && !ch.solve_pending) || (side_g && !ch.g_pending)) {
      // first step of this chain: the inputs of the two streams come from the chain's stream
      cudaEvent_t e = c->ev_sw[(c->ev_sw_next++) % BTA_NSW];
      CK(cudaEventRecord(e, lane(lch, st, lch ? ch.on_small : false)));
      if (side_solve && !ch.solve_pending) {
        CK(cudaStreamWaitEvent(ch.ss, e, 0));
        ch.solve_pending = true;
      }
      if (side_g && !ch.g_pending) {
        CK(cudaStreamWaitEvent(ch.gs, e, 0));
        ch.g_pending = true;
      }
    }
    if (nr > 0) {
      double* part = side_solve ? ch.part2 : ch.part;
      auto SV = [&]() { return side_solve ? ch.ss : lane(lch, st, true); };
      const double* z = ch.Rout + t * ch.rout_stride + (long long)zrow0 * ch.ld_rout;
      const double* u = z;
      int ld_u = ch.ld_rout;
      if (arrow) {
        CK(launch_small_left_mul(nr, a, b, ch.xT, a, LC, ld_lc, -1.0, 1.0, u, ld_u, ch.ubuf, b, SV()));
        BTA_COUNT(c);
        u = ch.ubuf;
        ld_u = b;
      }
      if (has_next) {
        const double* xnext = (t < nt - 1) ? ch.xout + (long long)ch.tg(t + 1) * b : ch.sep_x;
        CK(launch_skinny_nn(nr, b, b, xnext, (int)ch.ld_x, LB, b, 0, -1.0, 1.0, u, ld_u,
                            ch.ubuf, b, part, SV()));
        c->launches += 2;
        u = ch.ubuf;
        ld_u = b;
      }
      if (ch.fill) {  // - L_Ft^T x_s
        CK(launch_skinny_nn(nr, b, b, ch.fill->xs, (int)ch.fill->ld_xs, ch.fill->LF + t * ch.fill->lf_stride, b, 0, -1.0,
                            1.0, u, ld_u, ch.ubuf, b, part, SV()));
        c->launches += 2;
        u = ch.ubuf;
        ld_u = b;
      }
      CK(launch_skinny_nn(nr, b, b, u, ld_u, X, b, 1, 1.0, 0.0, nullptr, 0, ch.xout + tg * b, (int)ch.ld_x,
                          part, SV()));
      c->launches += 2;
    }
    if (!ch.selinv) return cudaSuccess;
    // (not in carry mode: there Z_B sits in the one L_B buffer that the next step rebuilds)
    const bool defer_tr = ch.contract && ch.rs && ch.pipe_ev && !ch.carry;
    if (defer_tr && ch.tr_armed[t & 1]) {  // Z_D / Z_C buffers of this parity: their traces (two steps ago) are done
      CK(cudaStreamWaitEvent(st, ch.pipe_ev[3 + (t & 1)], 0));
      if (ch.hi) CK(cudaStreamWaitEvent(ch.hi, ch.pipe_ev[3 + (t & 1)], 0));
    }
    // ---- selected inversion (R10), tensor-friendly form:  G = L_B X,  E = L_C X,
    //      Z_B = -Z_D{t+1} G - Z_C{t+1}^T E,  Z_C = -Z_C{t+1} G - Z_T E,  Z_D = X^T X - Z_B^T G - Z_C^T E
    double* ZDcur = (t & 1) ? ch.W2 : ch.W3;
    const double* ZDnext = (t < nt - 1) ? ((t & 1) ? ch.W3 : ch.W2) : ch.sep_ZD;
    double* ZCcur = ch.ZC[t & 1];
    const double* ZCnext = (t < nt - 1) ? ch.ZC[(t & 1) ^ 1] : ch.sep_ZC;
    double* Eb = ch.Ebuf;
    double* Yb = ch.Ybuf;
    cudaEvent_t ev_ey = nullptr;   // side_solve: E and Z_T E of this step are ready (recorded on the solve stream)
    if (arrow) {
      const bool side_ey = side_solve && ch.pipe_ev && ch.Ebuf2[t & 1] && ch.Ybuf2[t & 1];
      cudaStream_t es = SS;
      double* part = ch.part;
      if (side_ey) {
        Eb = ch.Ebuf2[t & 1];
        Yb = ch.Ybuf2[t & 1];
        es = ch.ss;
        part = ch.part2;
        if (ch.ey_used[t & 1]) CK(cudaStreamWaitEvent(es, ch.pipe_ev[7 + (t & 1)], 0));  // step t+2 is done with the slot
      }
      CK(launch_skinny_nn(a, b, b, LC, ld_lc, X, b, 1, 1.0, 0.0, nullptr, 0, Eb, b, part, es));  // E
      CK(launch_small_left_mul(a, a, b, ch.ZT, a, Eb, b, 1.0, 0.0, nullptr, 0, Yb, b, es));     // Z_T E
      c->launches += 3;
      if (side_ey) {
        ev_ey = ch.pipe_ev[5 + (t & 1)];
        CK(cudaEventRecord(ev_ey, es));
      }
    }
    Fill* fl = ch.fill;
    if (ev_ey) {  // the chain's lanes use E and Z_T E from here on
      CK(cudaStreamWaitEvent(st, ev_ey, 0));
      if (ch.hi && lch) CK(cudaStreamWaitEvent(ch.hi, ev_ey, 0));
    }
    double* LFt = fl ? fl->LF + t * fl->lf_stride : nullptr;
    if (fl) {  // H = L_F X;  the arrow term Z_T E gains Sigma[T,s] H
      CK(launch_gemm(G(GEMM_NN, b, b, b, 1.0, LFt, b, X, b, 0.0, fl->H, b, KLO_N0, KHI_K, OUT_FULL), SB));
      BTA_COUNT(c);
      if (arrow) {
        CK(launch_skinny_nn(a, b, b, fl->ZCs, b, fl->H, b, 0, 1.0, 1.0, Yb, b, Yb, b, ch.part, SS));
        c->launches += 2;
      }
    }
    if (has_next) {
      double* Gm = side_g ? ch.Gm2[t & 1] : ch.W1;
      if (side_g) {
        cudaStream_t gs = ch.gs;
        if (ch.g_used[t & 1]) CK(cudaStreamWaitEvent(gs, ch.pipe_ev[11 + (t & 1)], 0));   // step t+2 is done with the slot
        CK(launch_gemm(G(GEMM_NN, b, b, b, 1.0, LB, b, X, b, 0.0, Gm, b, KLO_N0, KHI_K, OUT_FULL), gs));
        // X^T X straight into this step's Z_D buffer: step t+1's Z_B product (and the traces of step t+2) have read it
        if (ch.zd_read[t & 1]) CK(cudaStreamWaitEvent(gs, ch.pipe_ev[13 + (t & 1)], 0));
        if (defer_tr && ch.tr_armed[t & 1]) CK(cudaStreamWaitEvent(gs, ch.pipe_ev[3 + (t & 1)], 0));
        CK(launch_gemm(G(GEMM_TN, b, b, b, 1.0, X, b, X, b, 0.0, ZDcur, b, KLO_M0, KHI_K, OUT_LOWER), gs));
        CK(cudaEventRecord(ch.pipe_ev[9 + (t & 1)], gs));
      } else {
        CK(launch_gemm(G(GEMM_NN, b, b, b, 1.0, LB, b, X, b, 0.0, Gm, b, KLO_N0, KHI_K, OUT_FULL), SB));
      }
      BTA_COUNT(c);
      if (side_solve) {  // the solve's reader of L_Bt has been issued (G's is covered by its ready event below)
        ev_solve = c->ev_sw[(c->ev_sw_next++) % BTA_NSW];
        CK(cudaEventRecord(ev_solve, ch.ss));
      }
      if (side_g) {
        CK(cudaStreamWaitEvent(st, ch.pipe_ev[9 + (t & 1)], 0));
        if (ch.hi && lch) CK(cudaStreamWaitEvent(ch.hi, ch.pipe_ev[9 + (t & 1)], 0));
      }
      if (arrow) {
        CK(launch_skinny_nn(a, b, b, ZCnext, b, Gm, b, 0, -1.0, -1.0, Yb, b, ZCcur, b, ch.part, SS));
        c->launches += 2;
      }
      double* ZB = LB;  // L_Bt is dead from here on: Z_Bt takes its slot
      if (ev_solve) CK(cudaStreamWaitEvent(SB, ev_solve, 0));
      CK(launch_gemm(G(GEMM_NN, b, b, b, -1.0, ZDnext, b, Gm, b, 0.0, ZB, b, KLO_ZERO, KHI_K, OUT_FULL), SB));
      BTA_COUNT(c);
      if (side_g) {  // the Z_D buffer of the other parity (Z_D{t+1}) may now receive X^T X of step t-1
        CK(cudaEventRecord(ch.pipe_ev[13 + ((t + 1) & 1)], SB));
        ch.zd_read[(t + 1) & 1] = true;
      }
      if (arrow) {
        CK(launch_gemm(G(GEMM_TN, b, b, a, -1.0, ZCnext, b, Eb, b, 1.0, ZB, b, KLO_ZERO, KHI_K, OUT_FULL), SB));
        BTA_COUNT(c);
      }
      if (!side_g)
        CK(launch_gemm(G(GEMM_TN, b, b, b, 1.0, X, b, X, b, 0.0, ZDcur, b, KLO_M0, KHI_K, OUT_LOWER), SB));
      if (fl) {
        // Sigma[s, t+1] is Z_F of the block below (stored [s][t+1]); below the last interior block it is the reduced
        // system's Sigma[e, s], stored the other way round
        const bool last = t == nt - 1;
        const double* ZFn = last ? fl->ZFe : fl->LF + (t + 1) * fl->lf_stride;
        //   Z_B -= Sigma[t+1, s] H
        CK(launch_gemm(G(last ? GEMM_NN : GEMM_TN, b, b, b, -1.0, ZFn, b, fl->H, b, 1.0, ZB, b, KLO_ZERO, KHI_K, OUT_FULL),
                       SB));
        //   Z_F = -(Sigma[s, t+1] G + Sigma[s,s] H + Sigma[T,s]^T E), into the slot of L_F (dead since H)
        CK(launch_gemm(G(last ? GEMM_TN : GEMM_NN, b, b, b, -1.0, ZFn, b, Gm, b, 0.0, LFt, b, KLO_ZERO, KHI_K, OUT_FULL),
                       SB));
        CK(launch_gemm(G(GEMM_NN, b, b, b, -1.0, fl->ZDs, b, fl->H, b, 1.0, LFt, b, KLO_ZERO, KHI_K, OUT_FULL), SB));
        if (arrow)
          CK(launch_gemm(G(GEMM_TN, b, b, a, -1.0, fl->ZCs, b, Eb, b, 1.0, LFt, b, KLO_ZERO, KHI_K, OUT_FULL), SB));
        //   Z_D -= Z_F^T H
        CK(launch_gemm(G(GEMM_TN, b, b, b, -1.0, LFt, b, fl->H, b, 1.0, ZDcur, b, KLO_ZERO, KHI_K, OUT_LOWER), SB));
        c->launches += arrow ? 5 : 4;
      }
      CK(launch_gemm(G(GEMM_TN, b, b, b, -1.0, ZB, b, Gm, b, 1.0, ZDcur, b, KLO_ZERO, KHI_K,
                       arrow ? OUT_LOWER : OUT_LOWER_MIRROR),
                     SB));
      c->launches += 2;
      if (side_g) {  // last reader of this step's G
        CK(cudaEventRecord(ch.pipe_ev[11 + (t & 1)], SB));
        ch.g_used[t & 1] = true;
      }
    } else {
      if (arrow) {
        scale_copy_kernel<<<(unsigned)(((long long)a * b + 255) / 256), 256, 0, SS>>>((long long)a * b, -1.0, Yb,
                                                                                      ZCcur);
        BTA_COUNT(c);
      }
      CK(launch_gemm(G(GEMM_TN, b, b, b, 1.0, X, b, X, b, 0.0, ZDcur, b, KLO_M0, KHI_K,
                       arrow ? OUT_LOWER : OUT_LOWER_MIRROR),
                     SB));
      BTA_COUNT(c);
    }
    if (arrow) {
      CK(launch_gemm(G(GEMM_TN, b, b, a, -1.0, ZCcur, b, Eb, b, 1.0, ZDcur, b, KLO_ZERO, KHI_K, OUT_LOWER_MIRROR),
                     SB));
      BTA_COUNT(c);
      if (ev_ey) {  // every use of this step's E / Z_T E has been issued in lane order
        CK(cudaEventRecord(ch.pipe_ev[7 + (t & 1)], lane(lch, st, lch ? ch.on_small : false)));
        ch.ey_used[t & 1] = true;
      }
    }
    if (ch.contract) {
      cudaStream_t ts = SS;
      if (defer_tr) {  // on the rows stream, after everything this step wrote
        cudaStream_t cur = lane(lch, st, lch ? ch.on_small : false);
        cudaEvent_t e = c->ev_sw[(c->ev_sw_next++) % BTA_NSW];
        CK(cudaEventRecord(e, cur));
        CK(cudaStreamWaitEvent(ch.rs, e, 0));
        ts = ch.rs;
      }
      CK(launch_trace_stencil(c, ch.chain, (int)tg, 0, ZDcur, b, ts));
      if (has_next && ch.tB(t) >= 0) CK(launch_trace_stencil(c, ch.chain, ch.tB(t), 1, LB, b, ts));
      if (fl && t == 0 && fl->tb_first >= 0) CK(launch_trace_stencil(c, ch.chain, fl->tb_first, 1, LFt, b, ts));
      if (arrow) CK(launch_noise_trace(c, (int)tg, ZDcur, b, ZCcur, b, ts));
      if (defer_tr) {
        CK(cudaEventRecord(ch.pipe_ev[3 + (t & 1)], ch.rs));
        ch.tr_armed[t & 1] = true;
        ch.rows_pending = true;
      }
    }
    if (ch.selinv_inplace) {
      CK(cudaMemcpyAsync(ch.Dp(t), ZDcur, bb * sizeof(double), cudaMemcpyDeviceToDevice, SB));
      if (arrow && ch.Cout)
        CK(cudaMemcpyAsync(ch.Cout + t * ch.cout_stride, ZCcur, (size_t)a * b * sizeof(double),
                           cudaMemcpyDeviceToDevice, SB));
    }
  }
  return cudaSuccess;
}

cudaError_t chain_backward(Chain& ch, cudaStream_t st) {
  for (int t = ch.nt - 1; t >= 0; --t) CK(chain_backward_step(ch, t, st));
  return cudaSuccess;
}
