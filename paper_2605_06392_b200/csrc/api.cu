// The C-ABI entry points of include/bta.h: argument checks, workspace carving, stream/event plumbing.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>

#include "api_util.h"

namespace {

struct ChainWs {
  double *D, *B, *W1, *W2, *W3, *Rin, *Rout, *ubuf, *Ebuf, *Ybuf, *ZC0, *ZC1, *part, *x, *dvec, *T, *rtip, *Xs, *LBs, *Bs;
};

// Workspace of one chain of the fused gradient.  Q_c: nt D slots, nt B slots (L_Bt is written one slot below
// B_t, so no copy), 3 scratch blocks, the arrow/rhs stacks; Q_p: the same without the stacks.
ChainWs carve_chain(Bump& bp, const ModelDims& md, bool cond, int store_mode) {
  ChainWs w{};
  const size_t bb = (size_t)md.b * md.b;
  const int P = md.a + 1;
  w.D = bp.take(bb * md.nt);
  if (store_mode != BTA_STORE_FACTOR) {
    w.Xs = bp.take(bb);
    w.LBs = bp.take(bb);
    w.Bs = bp.take(bb);
  } else {
    w.B = bp.take(bb * md.nt);
  }
  w.W1 = bp.take(bb);
  w.W2 = bp.take(bb);
  w.W3 = bp.take(bb);
  w.dvec = bp.take(md.N);
  w.T = bp.take(md.a * md.a);
  if (cond) {
    w.Rin = bp.take((size_t)md.nt * P * md.b);
    w.Rout = bp.take((size_t)md.nt * P * md.b);
    w.ubuf = bp.take(md.b);
    w.Ebuf = bp.take((size_t)md.a * md.b);
    w.Ybuf = bp.take((size_t)md.a * md.b);
    w.ZC0 = bp.take((size_t)md.a * md.b);
    w.ZC1 = bp.take((size_t)md.a * md.b);
    w.part = bp.take(skinny_nn_part_doubles(P, md.b, md.b));
    w.x = bp.take(md.N);
    w.rtip = bp.take(md.a);
  }
  return w;
}

size_t grad_ws_bytes(const ModelDims& md, int store_mode) {
  Bump bp(nullptr);
  carve_chain(bp, md, true, store_mode);
  carve_chain(bp, md, false, store_mode);
  return bp.off + 256;
}

struct OpWs {
  double *W1, *W2, *W3, *Rtmp, *zbuf, *ubuf, *Ebuf, *Ybuf, *ZC0, *ZC1, *part, *dvec, *Tt, *xT, *scal;
};
constexpr int SOLVE_CHUNK = 8;

OpWs carve_op(Bump& bp, const ModelDims& md) {
  OpWs w{};
  const size_t bb = (size_t)md.b * md.b;
  w.W1 = bp.take(bb);
  w.W2 = bp.take(bb);
  w.W3 = bp.take(bb);
  w.Rtmp = bp.take((size_t)(AMAX + 1) * md.b);
  w.zbuf = bp.take((size_t)SOLVE_CHUNK * md.N);
  w.ubuf = bp.take((size_t)SOLVE_CHUNK * md.b);
  w.Ebuf = bp.take((size_t)md.a * md.b);
  w.Ybuf = bp.take((size_t)md.a * md.b);
  w.ZC0 = bp.take((size_t)md.a * md.b);
  w.ZC1 = bp.take((size_t)md.a * md.b);
  w.part = bp.take(skinny_nn_part_doubles(AMAX + 1, md.b, md.b));
  w.dvec = bp.take(md.N);
  w.Tt = bp.take((size_t)md.a * (md.a + SOLVE_CHUNK));
  w.xT = bp.take((size_t)SOLVE_CHUNK * md.a);
  w.scal = bp.take(8);
  return w;
}

int check_pivot(bta_ctx* c, cudaStream_t st) {
  unsigned long long flag = 0;
  BTA_CUDA_OK(cudaMemcpyAsync(&flag, c->pivot_flag, sizeof flag, cudaMemcpyDeviceToHost, st));
  BTA_CUDA_OK(cudaStreamSynchronize(st));
  if (flag != ~0ull) {
    c->last_pivot = (long long)flag;
    char buf[160];
    snprintf(buf, sizeof buf, "matrix is not positive definite: first non-positive pivot at global row %lld",
             (long long)flag);
    bta_set_error(buf);
    return BTA_ERR_NOTSPD;
  }
  c->last_pivot = 0;
  return BTA_OK;
}

}  // namespace

extern "C" size_t bta_workspace_bytes_op(const bta_ctx* c) {
  if (!c) return 0;
  Bump bp(nullptr);
  carve_op(bp, c->md);
  return bp.off + 256;
}

extern "C" int bta_assemble(bta_ctx* c, const double* theta, int which, bta_blocks out, void* stream) {
  if (!c || !theta) return bad("bta_assemble: null ctx or theta");
  if (which != BTA_PRIOR && which != BTA_COND) return bad("bta_assemble: which must be BTA_PRIOR or BTA_COND");
  if (!out.D || (c->md.nt > 1 && !out.B) || !out.T) return bad("bta_assemble: D, B and T are required");
  cudaStream_t st = (cudaStream_t)stream;
  const ModelDims& md = c->md;
  DeviceGuard guard(c->device);
  memcpy(c->host_pinned, theta, md.d * sizeof(double));
  BTA_CUDA_OK(cudaMemcpyAsync(c->theta_dev, c->host_pinned, md.d * sizeof(double), cudaMemcpyHostToDevice, st));
  BTA_CUDA_OK(launch_theta_prep(c, st));
  const long long bb = (long long)md.b * md.b;
  BTA_CUDA_OK(launch_assemble(c, which, out.D, bb, out.B, bb, out.C, (long long)md.a * md.b, out.T, md.a, out.rhs, md.b,
                              out.rhs ? out.rhs + (long long)md.nt * md.b : nullptr, 1, st));
  BTA_CUDA_OK(cudaStreamSynchronize(st));  // host_pinned is reused by the next call
  return BTA_OK;
}

extern "C" int bta_factor_logdet(bta_ctx* c, bta_blocks io, int which, double* logdet, double* diagL, void* ws,
                                 void* stream) {
  if (!c || !ws) return bad("bta_factor_logdet: null ctx or workspace");
  if (which != BTA_PRIOR && which != BTA_COND) return bad("bta_factor_logdet: bad `which`");
  if (!io.D || (c->md.nt > 1 && !io.B) || !io.T || (which == BTA_COND && !io.C))
    return bad("bta_factor_logdet: D, B, T (and C for BTA_COND) are required");
  cudaStream_t st = (cudaStream_t)stream;
  const ModelDims& md = c->md;
  DeviceGuard guard(c->device);
  Bump bp(ws);
  OpWs w = carve_op(bp, md);
  SmallLayout L = small_layout(md);
  const int chs = which == BTA_COND ? CH_COND : CH_PRIOR;
  BTA_CUDA_OK(cudaMemsetAsync(c->pivot_flag, 0xFF, sizeof(unsigned long long), st));
  Chain ch;
  ch.c = c;
  ch.chain = chs;
  ch.b = md.b;
  ch.nt = md.nt;
  ch.a = md.a;
  ch.nr = 0;
  ch.zero_upper = true;
  ch.arrow_rows = which == BTA_COND;
  ch.D = io.D;
  ch.d_stride = (long long)md.b * md.b;
  ch.Bin = ch.Bout = io.B;
  ch.b_stride = ch.d_stride;
  ch.Rin = ch.Rout = io.C;
  ch.rin_stride = ch.rout_stride = (long long)md.a * md.b;
  ch.ld_rin = ch.ld_rout = md.b;
  ch.Rtmp = w.Rtmp;
  ch.T = io.T;
  ch.ldT = md.a;
  ch.W1 = w.W1;
  ch.W2 = w.W2;
  ch.W3 = w.W3;
  ch.part = w.part;
  ch.dvec = diagL ? diagL : w.dvec;
  ch.Tt = w.Tt;
  ch.LT = io.T;
  ch.ZT = c->small + L.ZT[chs];
  BTA_CUDA_OK(chain_forward(ch, st));
  // Rout == Rin for t = 0 would alias in the second stack product only when t > 0 uses Rtmp: fine (see sweep.cu)
  BTA_CUDA_OK(launch_logdet_partial(c, chs, ch.dvec, st));
  BTA_CUDA_OK(launch_logdet_final(c, chs, w.scal, st));
  BTA_CUDA_OK(cudaMemcpyAsync(c->host_pinned, w.scal, sizeof(double), cudaMemcpyDeviceToHost, st));
  int rc = check_pivot(c, st);
  if (logdet) *logdet = c->host_pinned[0];
  return rc;
}

// include/bta_diag.h: the block factorisation of the forward sweeps alone (kernel tests and timing)
extern "C" int bta_diag_potrf_inv(bta_ctx* c, double* A, int ld, int n, double* T1, double* T2, double* diagL,
                                  void* stream) {
  if (!c || !A || n <= 0 || ld < n) return bad("bta_diag_potrf_inv: null ctx or block, or bad sizes");
  if (n > leaf_max_n() && (!T1 || !T2))
    return bad("bta_diag_potrf_inv: blocks above 144 rows need the scratch blocks T1, T2");
  cudaStream_t st = (cudaStream_t)stream;
  DeviceGuard guard(c->device);
  BTA_CUDA_OK(cudaMemsetAsync(c->pivot_flag, 0xFF, sizeof(unsigned long long), st));
  BTA_CUDA_OK(potrf_inv(c, nullptr, A, ld, 0, n, T1, T2, diagL, 0, st));
  return check_pivot(c, st);
}

extern "C" int bta_solve(bta_ctx* c, bta_blocks Lf, int which, double* rhs, int nrhs, void* ws, void* stream) {
  if (!c || !ws || !rhs) return bad("bta_solve: null ctx, workspace or rhs");
  if (which != BTA_PRIOR && which != BTA_COND) return bad("bta_solve: bad `which`");
  if (nrhs < 0) return bad("bta_solve: nrhs < 0");
  if (!Lf.D || (c->md.nt > 1 && !Lf.B) || !Lf.T || (which == BTA_COND && !Lf.C)) return bad("bta_solve: missing factor");
  cudaStream_t st = (cudaStream_t)stream;
  const ModelDims& md = c->md;
  DeviceGuard guard(c->device);
  Bump bp(ws);
  OpWs w = carve_op(bp, md);
  for (int r0 = 0; r0 < nrhs; r0 += SOLVE_CHUNK) {
    const int nr = std::min(SOLVE_CHUNK, nrhs - r0);
    double* R = rhs + (long long)r0 * md.N;
    Chain ch;
    ch.c = c;
    ch.b = md.b;
    ch.nt = md.nt;
    ch.a = md.a;
    ch.nr = nr;
    ch.factor_blocks = false;
    ch.tip_chol = false;
    ch.arrow_given = which == BTA_COND;
    ch.LCgiven = Lf.C;
    ch.lc_stride = (long long)md.a * md.b;
    ch.D = Lf.D;
    ch.d_stride = (long long)md.b * md.b;
    ch.Bin = ch.Bout = Lf.B;
    ch.b_stride = ch.d_stride;
    ch.Rin = R;
    ch.rin_stride = md.b;
    ch.ld_rin = (int)md.N;
    ch.Rout = w.zbuf;
    ch.rout_stride = md.b;
    ch.ld_rout = (int)md.N;
    ch.Rtmp = w.Rtmp;
    ch.T = Lf.T;
    ch.ldT = md.a;
    ch.rhs_tip = R + (long long)md.nt * md.b;
    ch.rhs_tip_stride = (int)md.N;
    ch.W1 = w.W1;
    ch.W2 = w.W2;
    ch.W3 = w.W3;
    ch.part = w.part;
    ch.ubuf = w.ubuf;
    ch.Tt = w.Tt;
    ch.LT = Lf.T;
    ch.xT = w.xT;
    ch.xout = R;
    ch.ld_x = md.N;
    BTA_CUDA_OK(chain_forward(ch, st));
    BTA_CUDA_OK(chain_backward(ch, st));
    BTA_CUDA_OK(cudaMemcpy2DAsync(R + (long long)md.nt * md.b, md.N * sizeof(double), w.xT, md.a * sizeof(double),
                                  md.a * sizeof(double), nr, cudaMemcpyDeviceToDevice, st));
  }
  BTA_CUDA_OK(cudaStreamSynchronize(st));
  return BTA_OK;
}

extern "C" int bta_selinv(bta_ctx* c, bta_blocks io, int which, void* ws, void* stream) {
  if (!c || !ws) return bad("bta_selinv: null ctx or workspace");
  if (which != BTA_PRIOR && which != BTA_COND) return bad("bta_selinv: bad `which`");
  if (!io.D || (c->md.nt > 1 && !io.B) || !io.T || (which == BTA_COND && !io.C)) return bad("bta_selinv: missing factor");
  cudaStream_t st = (cudaStream_t)stream;
  const ModelDims& md = c->md;
  DeviceGuard guard(c->device);
  Bump bp(ws);
  OpWs w = carve_op(bp, md);
  SmallLayout L = small_layout(md);
  const int chs = which == BTA_COND ? CH_COND : CH_PRIOR;
  Chain ch;
  ch.c = c;
  ch.chain = chs;
  ch.b = md.b;
  ch.nt = md.nt;
  ch.a = md.a;
  ch.factor_blocks = false;
  ch.selinv = true;
  ch.selinv_inplace = true;
  ch.arrow_given = which == BTA_COND;
  ch.LCgiven = io.C;
  ch.lc_stride = (long long)md.a * md.b;
  ch.Cout = io.C;
  ch.cout_stride = ch.lc_stride;
  ch.D = io.D;
  ch.d_stride = (long long)md.b * md.b;
  ch.Bin = ch.Bout = io.B;
  ch.b_stride = ch.d_stride;
  ch.W1 = w.W1;
  ch.W2 = w.W2;
  ch.W3 = w.W3;
  ch.part = w.part;
  ch.Ebuf = w.Ebuf;
  ch.Ybuf = w.Ybuf;
  ch.ZC[0] = w.ZC0;
  ch.ZC[1] = w.ZC1;
  ch.ZT = c->small + L.ZT[chs];
  BTA_CUDA_OK(launch_tip_inverse(io.T, md.a, ch.ZT, st));
  BTA_COUNT(c);
  BTA_CUDA_OK(chain_backward(ch, st));
  BTA_CUDA_OK(cudaMemcpyAsync(io.T, ch.ZT, sizeof(double) * md.a * md.a, cudaMemcpyDeviceToDevice, st));
  BTA_CUDA_OK(cudaStreamSynchronize(st));
  return BTA_OK;
}

// ------------------------------------------------------------------------------------------------
// The hot path: f(theta), grad f(theta)   (PAPER.md:44 Eq. 1, :121 Eq. 6)
// ------------------------------------------------------------------------------------------------
namespace {

// Enqueue one whole gradient: theta upload -> both chains (interleaved on s0 / s1) -> scalar assembly -> result
// download into pinned host memory.  With `timed` the stage events are recorded (not capturable in a graph).
int enqueue_gradient(bta_ctx* c, void* ws, cudaStream_t s0, cudaStream_t s1, bool timed, bool value_only) {
  const ModelDims& md = c->md;
  const bool serial = (s0 == s1);
  Bump bp(ws);
  const bool carry = c->store_mode != BTA_STORE_FACTOR;  // host staging needs the two-way sweep (nt >= 3): plain carry here
  ChainWs wc = carve_chain(bp, md, true, c->store_mode);
  ChainWs wp = carve_chain(bp, md, false, c->store_mode);
  SmallLayout L = small_layout(md);
  const long long bb = (long long)md.b * md.b;
  const int P = md.a + 1;
  cudaEvent_t* ev = c->ev;
#define REC(i, st)                                    \
  do {                                                \
    if (timed) BTA_CUDA_OK(cudaEventRecord(ev[i], st)); \
  } while (0)

  REC(0, s0);
  BTA_CUDA_OK(cudaMemcpyAsync(c->theta_dev, c->host_pinned, md.d * sizeof(double), cudaMemcpyHostToDevice, s0));
  BTA_CUDA_OK(launch_theta_prep(c, s0));
  BTA_CUDA_OK(cudaMemsetAsync(c->pivot_flag, 0xFF, sizeof(unsigned long long), s0));
  BTA_CUDA_OK(cudaEventRecord(ev[9], s0));
  if (!serial) BTA_CUDA_OK(cudaStreamWaitEvent(s1, ev[9], 0));

  // ---- Q_c chain on s0 ----
  Chain cc;
  cc.c = c;
  cc.chain = CH_COND;
  cc.b = md.b;
  cc.nt = md.nt;
  cc.a = md.a;
  cc.nr = 1;
  cc.arrow_rows = true;
  cc.selinv = cc.contract = !value_only;
  cc.D = wc.D;
  cc.d_stride = bb;
  cc.carry = carry;
  cc.which = BTA_COND;
  cc.Xs = wc.Xs;
  cc.LBs = wc.LBs;
  cc.Bs = wc.Bs;
  cc.Bin = carry ? nullptr : wc.B + bb;  // B_t assembled into slot t+1, L_Bt written to slot t
  cc.Bout = wc.B;
  cc.b_stride = bb;
  cc.Rin = wc.Rin;
  cc.rin_stride = (long long)P * md.b;
  cc.ld_rin = md.b;
  cc.Rout = wc.Rout;
  cc.rout_stride = (long long)P * md.b;
  cc.ld_rout = md.b;
  cc.Rtmp = nullptr;
  cc.T = wc.T;
  cc.ldT = md.a;
  cc.rhs_tip = wc.rtip;
  cc.rhs_tip_stride = md.a;
  cc.W1 = wc.W1;
  cc.W2 = wc.W2;
  cc.W3 = wc.W3;
  cc.part = wc.part;
  cc.ubuf = wc.ubuf;
  cc.Ebuf = wc.Ebuf;
  cc.Ybuf = wc.Ybuf;
  cc.ZC[0] = wc.ZC0;
  cc.ZC[1] = wc.ZC1;
  cc.dvec = wc.dvec;
  cc.Tt = c->small + L.Tt[CH_COND];
  cc.LT = c->small + L.LT[CH_COND];
  cc.zT = c->small + L.zT[CH_COND];
  cc.xT = c->small + L.xT[CH_COND];
  cc.ZT = c->small + L.ZT[CH_COND];
  cc.xout = wc.x;
  cc.ld_x = md.N;

  // ---- Q_p chain (Phase C) on the side stream ----
  Chain cp;
  cp.c = c;
  cp.chain = CH_PRIOR;
  cp.b = md.b;
  cp.nt = md.nt;
  cp.a = md.a;
  cp.nr = 0;
  cp.selinv = cp.contract = !value_only;
  cp.D = wp.D;
  cp.d_stride = bb;
  cp.carry = carry;
  cp.which = BTA_PRIOR;
  cp.Xs = wp.Xs;
  cp.LBs = wp.LBs;
  cp.Bs = wp.Bs;
  cp.Bin = carry ? nullptr : wp.B + bb;
  cp.Bout = wp.B;
  cp.b_stride = bb;
  cp.T = wp.T;
  cp.ldT = md.a;
  cp.W1 = wp.W1;
  cp.W2 = wp.W2;
  cp.W3 = wp.W3;
  cp.dvec = wp.dvec;
  cp.Tt = c->small + L.Tt[CH_PRIOR];
  cp.LT = c->small + L.LT[CH_PRIOR];
  cp.ZT = c->small + L.ZT[CH_PRIOR];

  // The two chains are independent (they meet only in the scalar assembly).  Their launches are interleaved
  // block by block from this one host thread so that both streams always have work queued: the latency-bound
  // parts of one chain (POTRF leaves, skinny kernels) overlap the GEMMs of the other.
  BTA_CUDA_OK(launch_assemble(c, BTA_COND, cc.D, bb, cc.Bin, bb, wc.Rin, cc.rin_stride, wc.T, md.a,
                              wc.Rin + (long long)md.a * md.b, cc.rin_stride, wc.rtip, 1, s0));
  REC(1, s0);
  REC(4, s1);
  BTA_CUDA_OK(launch_assemble(c, BTA_PRIOR, cp.D, bb, cp.Bin, bb, nullptr, 0, wp.T, md.a, nullptr, 0, nullptr, 0, s1));
  REC(5, s1);
  BTA_CUDA_OK(chain_forward_begin(cc, s0));
  BTA_CUDA_OK(chain_forward_begin(cp, s1));
  for (int t = 0; t < md.nt; ++t) {
    BTA_CUDA_OK(chain_forward_step(cc, t, s0));
    BTA_CUDA_OK(chain_forward_step(cp, t, s1));
  }
  BTA_CUDA_OK(chain_forward_end(cc, s0));
  BTA_CUDA_OK(launch_logdet_partial(c, CH_COND, wc.dvec, s0));
  REC(2, s0);
  BTA_CUDA_OK(chain_forward_end(cp, s1));
  BTA_CUDA_OK(launch_logdet_partial(c, CH_PRIOR, wp.dvec, s1));
  REC(6, s1);
  for (int t = md.nt - 1; t >= 0; --t) {
    BTA_CUDA_OK(chain_backward_step(cc, t, s0));                  // value only: just the upper solve (Eqs. 3-5)
    if (!value_only) BTA_CUDA_OK(chain_backward_step(cp, t, s1));
  }
  BTA_CUDA_OK(cudaMemcpyAsync(wc.x + (long long)md.nt * md.b, cc.xT, md.a * sizeof(double), cudaMemcpyDeviceToDevice,
                              s0));
  BTA_CUDA_OK(launch_quad_stencil(c, wc.x, s0));
  BTA_CUDA_OK(launch_residual(c, wc.x, s0));
  REC(3, s0);
  BTA_CUDA_OK(cudaEventRecord(ev[7], s1));
  if (!serial) BTA_CUDA_OK(cudaStreamWaitEvent(s0, ev[7], 0));

  // ---- scalar assembly (a9) ----
  REC(10, s0);
  BTA_CUDA_OK(launch_scalars(c, s0));
  const int nout = 1 + md.d + 2 + 3 * md.d + md.k + 1;
  BTA_CUDA_OK(cudaMemcpyAsync(c->host_pinned + 64, c->small + L.out, nout * sizeof(double), cudaMemcpyDeviceToHost,
                              s0));
  BTA_CUDA_OK(cudaMemcpyAsync(c->x_keep, wc.x, md.N * sizeof(double), cudaMemcpyDeviceToDevice, s0));
  REC(8, s0);
  c->have_x = true;
#undef REC
  return BTA_OK;
}

// ------------------------------------------------------------------------------------------------
// Two-way (twisted) elimination: time-domain partitioning with P = 2 inside one GPU (PAPER.md:175-183,
// SURVEY.md §8(f) NEXT-3, first step).  Blocks 0..h-1 are eliminated upwards and blocks nt-1..h+1 downwards
// (the same chain code on the time-reversed sub-matrix with transposed coupling blocks); both meet at the
// separator block h, which is eliminated last together with the arrow tip.  No fill-in, the same flops, the
// same results up to rounding order -- but four independent chains (two per matrix) instead of two, so the
// latency-bound POTRF phases of one chain overlap the GEMMs of three others.
struct SubWs {
  double *B, *W1, *W2, *W3, *Xs, *LBs, *Bs, *ubuf, *Ebuf, *Ybuf, *ZC0, *ZC1, *part, *part2, *EY2, *G2, *ring;
};
constexpr int AHEAD_MAXB = 1024;   // block sizes whose backward steps run G, X^T X, the solve and E ahead of the chain
constexpr int HOST_RING = 4;  // device slots per sub-chain for the diagonal blocks in BTA_STORE_HOST
struct MatWs {
  double *D, *dvec, *T, *Rin, *Rout, *x, *rtip, *Tt2;
  SubWs sub[3];  // up, down, separator
};

int twist_h(const ModelDims& md) { return md.nt / 2; }

MatWs carve_twist(Bump& bp, const ModelDims& md, bool cond, int store_mode) {
  MatWs w{};
  const size_t bb = (size_t)md.b * md.b;
  const int P = md.a + 1, h = twist_h(md);
  const int len[3] = {h, md.nt - 1 - h, 1};
  w.D = bp.take(store_mode == BTA_STORE_HOST ? bb : bb * md.nt);  // host staging: only the separator block
  w.dvec = bp.take(md.N);
  w.T = bp.take(md.a * md.a);
  w.Tt2 = bp.take(md.a * (md.a + 1));
  if (cond) {
    w.Rin = bp.take((size_t)md.nt * P * md.b);
    w.Rout = bp.take((size_t)md.nt * P * md.b);
    w.x = bp.take(md.N);
    w.rtip = bp.take(md.a);
  }
  for (int q = 0; q < 3; ++q) {
    SubWs& s = w.sub[q];
    s.W1 = bp.take(bb);
    s.W2 = bp.take(bb);
    s.W3 = bp.take(bb);
    if (q < 2) {
      if (store_mode != BTA_STORE_FACTOR) {
        s.Xs = bp.take(bb);
        s.LBs = bp.take(bb);
        s.Bs = bp.take(bb);
        if (store_mode == BTA_STORE_HOST) s.ring = bp.take(bb * HOST_RING);
      } else {
        s.B = bp.take(bb * (len[q] + 1));
        if (md.b <= AHEAD_MAXB) s.G2 = bp.take(2 * bb);   // ring of two G = L_B X (sweep.h: Chain::Gm2)
      }
    }
    if (cond) {
      s.ubuf = bp.take(md.b);
      s.Ebuf = bp.take((size_t)md.a * md.b);
      s.Ybuf = bp.take((size_t)md.a * md.b);
      s.ZC0 = bp.take((size_t)md.a * md.b);
      s.ZC1 = bp.take((size_t)md.a * md.b);
      s.part = bp.take(skinny_nn_part_doubles(P, md.b, md.b));
      // the solve stream's own partial sums (upper solve: 1 row; arrow product E: a rows) and its ring of E / Z_T E
      s.part2 = bp.take(skinny_nn_part_doubles(std::max(1, md.a), md.b, md.b));
      s.EY2 = bp.take((size_t)4 * md.a * md.b);
    }
  }
  return w;
}

size_t twist_ws_bytes(const ModelDims& md, int store_mode) {
  Bump bp(nullptr);
  carve_twist(bp, md, true, store_mode);
  carve_twist(bp, md, false, store_mode);
  return bp.off + 256;
}

bool use_twist(const bta_ctx* c) { return c->opt.twist != 0 && c->md.nt >= 3; }

// The three chains (up, down, separator) of one matrix.
void make_twist_chains(bta_ctx* c, const MatWs& w, bool cond, bool value_only, Chain ch[3]) {
  const ModelDims& md = c->md;
  SmallLayout L = small_layout(md);
  const long long bb = (long long)md.b * md.b;
  const int P = md.a + 1, h = twist_h(md);
  const int chs = cond ? CH_COND : CH_PRIOR;
  const bool carry = c->store_mode != BTA_STORE_FACTOR, host = c->store_mode == BTA_STORE_HOST;
  const long long rs = (long long)P * md.b;
  for (int q = 0; q < 3; ++q) {
    Chain& k = ch[q];
    const SubWs& s = w.sub[q];
    k = Chain();
    k.c = c;
    k.chain = chs;
    k.which = cond ? BTA_COND : BTA_PRIOR;
    k.b = md.b;
    k.a = md.a;
    k.nr = cond ? 1 : 0;
    k.arrow_rows = cond;
    k.selinv = k.contract = !value_only;
    k.nt = q == 0 ? h : (q == 1 ? md.nt - 1 - h : 1);
    k.t0 = q == 0 ? 0 : (q == 1 ? md.nt - 1 : h);
    k.tdir = q == 1 ? -1 : 1;
    k.tail_coupling = q < 2;
    k.transposeB = q == 1;
    k.tt_zero = q == 1;
    k.carry = carry && q < 2;
    k.D = w.D + (long long)k.t0 * bb;
    k.d_stride = k.tdir * bb;
    if (host) {
      k.D = q < 2 ? s.ring : w.D;
      k.d_stride = bb;
      if (q < 2) {
        const int mi = cond ? 0 : 1;
        k.ring = HOST_RING;
        k.hostD = c->host_buf + ((long long)mi * (md.nt - 1) + (q == 1 ? h : 0)) * bb;
        k.cs = c->s_copy[2 * mi + q];
        k.ring_ev = c->ev_ring[2 * mi + q];
      }
    }
    k.Bin = (q < 2 && !carry) ? s.B + bb : nullptr;
    k.Bout = s.B;
    k.b_stride = bb;
    k.Xs = s.Xs;
    k.LBs = s.LBs;
    k.Bs = s.Bs;
    if (cond) {
      k.Rin = w.Rin + (long long)k.t0 * rs;
      k.rin_stride = k.tdir * rs;
      k.ld_rin = md.b;
      k.Rout = w.Rout + (long long)k.t0 * rs;
      k.rout_stride = k.tdir * rs;
      k.ld_rout = md.b;
      k.rhs_tip = w.rtip;
      k.rhs_tip_stride = md.a;
      k.ubuf = s.ubuf;
      k.Ebuf = s.Ebuf;
      k.Ybuf = s.Ybuf;
      k.ZC[0] = s.ZC0;
      k.ZC[1] = s.ZC1;
      k.part = s.part;
      k.part2 = s.part2;
      for (int r = 0; r < 2; ++r) {
        k.Ebuf2[r] = s.EY2 + (size_t)(2 * r) * md.a * md.b;
        k.Ybuf2[r] = s.EY2 + (size_t)(2 * r + 1) * md.a * md.b;
      }
      k.xout = w.x;
      k.ld_x = md.N;
    }
    k.T = w.T;
    k.ldT = md.a;
    k.W1 = s.W1;
    if (s.G2) {
      k.Gm2[0] = s.G2;
      k.Gm2[1] = s.G2 + bb;
    }
    k.W2 = s.W2;
    k.W3 = s.W3;
    k.dvec = w.dvec;
    k.Tt = q == 1 ? w.Tt2 : c->small + L.Tt[chs];
    k.LT = c->small + L.LT[chs];
    k.zT = c->small + L.zT[chs];
    k.xT = c->small + L.xT[chs];
    k.ZT = c->small + L.ZT[chs];
  }
  // what the sub-chains see as their "next" block in the backward sweep: the separator
  for (int q = 0; q < 2; ++q) {
    ch[q].sep_x = cond ? w.x + (long long)h * md.b : nullptr;
    ch[q].sep_ZD = ch[2].W3;      // Z_D of local block 0 of the separator chain (t & 1 == 0 -> W3)
    ch[q].sep_ZC = ch[2].ZC[0];
  }
}

int enqueue_gradient_twisted(bta_ctx* c, void* ws, cudaStream_t s0, bool timed, bool value_only) {
  const ModelDims& md = c->md;
  Bump bp(ws);
  MatWs wc = carve_twist(bp, md, true, c->store_mode);
  MatWs wp = carve_twist(bp, md, false, c->store_mode);
  SmallLayout L = small_layout(md);
  const long long bb = (long long)md.b * md.b;
  const int P = md.a + 1, h = twist_h(md);
  const bool carry = c->store_mode != BTA_STORE_FACTOR, host = c->store_mode == BTA_STORE_HOST;
  if (host && (!c->host_buf || c->host_bytes < bta_host_bytes(c)))
    return bad("inla_value_and_grad: BTA_STORE_HOST needs bta_set_host_buffer(ctx, pinned, bta_host_bytes(ctx)) first");
  cudaEvent_t* ev = c->ev;
  // streams: [matrix][up, down]
  cudaStream_t st[2][2] = {{s0, c->s_aux[0]}, {c->s_side, c->s_aux[1]}};
#define REC(i, s)                                      \
  do {                                                 \
    if (timed) BTA_CUDA_OK(cudaEventRecord(ev[i], s)); \
  } while (0)

  REC(0, s0);
  BTA_CUDA_OK(cudaMemcpyAsync(c->theta_dev, c->host_pinned, md.d * sizeof(double), cudaMemcpyHostToDevice, s0));
  BTA_CUDA_OK(launch_theta_prep(c, s0));
  BTA_CUDA_OK(cudaMemsetAsync(c->pivot_flag, 0xFF, sizeof(unsigned long long), s0));
  BTA_CUDA_OK(cudaEventRecord(ev[9], s0));
  BTA_CUDA_OK(cudaStreamWaitEvent(st[1][0], ev[9], 0));

  Chain ch[2][3];  // [0] = Q_c, [1] = Q_p (Phase C)
  make_twist_chains(c, wc, true, value_only, ch[0]);
  make_twist_chains(c, wp, false, value_only, ch[1]);
  const MatWs* W[2] = {&wc, &wp};
  {
    const int lanes = c->opt.lanes;
    if (lanes)
      for (int m = 0; m < 2; ++m) {
        ch[m][0].hi = c->s_hi[2 * m];
        ch[m][1].hi = c->s_hi[2 * m + 1];
        ch[m][2].hi = c->s_hi[2 * m];  // the separator runs on the up chain's streams
        for (int q = 0; q < 3; ++q) ch[m][q].lanes_bwd = lanes != 2;
      }
  }
  auto join_lanes = [&](int m, int q) { return chain_to_big(ch[m][q], st[m][q == 2 ? 0 : q]); };
  for (int m = 0; m < 2; ++m)
    for (int q = 0; q < 3; ++q) ch[m][q].trace_id = 3 * m + q;
  // side streams: off-chain work of the coupled forward step (b <= 1024); the events of the pipelined forward steps
  for (int m = 0; m < 2; ++m)
    for (int q = 0; q < 2; ++q) {
      if (c->opt.split) ch[m][q].xs = c->s_x[2 * m + q];
      ch[m][q].pipe_ev = c->ev_pipe[2 * m + q];
      // rows stream: pays where a step is latency-bound (measured: config 0 -11 %, config 1 -10 %; at b = 2304 the
      // extra concurrency costs 3 %), so only up to the size where the whole gradient is graph-replayed
      if (c->opt.rows && md.b <= 1024) ch[m][q].rs = c->s_r[2 * m + q];
      // solve stream (the forward steps' side stream is idle in the backward sweep): same size rule
      if (c->opt.rows && md.b <= AHEAD_MAXB && !carry) {
        ch[m][q].ss = c->s_x[2 * m + q];
        ch[m][q].gs = c->s_g[2 * m + q];
      }
    }

  // ---- assemble: D (all blocks), arrow/rhs rows, tip on the up stream; coupling blocks per sub-chain
  // The diagonal blocks are assembled lazily, a few blocks ahead of each sub-chain (assemble_ahead below): the 2 nt
  // blocks are 69 GB of writes that would otherwise sit in front of the first POTRF.
  BTA_CUDA_OK(launch_assemble(c, BTA_COND, nullptr, bb, nullptr, 0, wc.Rin, (long long)P * md.b, wc.T, md.a,
                              wc.Rin + (long long)md.a * md.b, (long long)P * md.b, wc.rtip, 1, st[0][0]));
  REC(4, st[1][0]);
  BTA_CUDA_OK(launch_assemble(c, BTA_PRIOR, nullptr, bb, nullptr, 0, nullptr, 0, wp.T, md.a, nullptr, 0, nullptr, 0,
                              st[1][0]));
  constexpr int AHEAD = 8;
  // local blocks [lo, hi) of sub-chain (m, q); the up chain also owns the separator (local index nt_up)
  auto assemble_range = [&](int m, int q, int lo, int hi) -> int {
    const Chain& k = ch[m][q];
    const int top = k.nt + (q == 0 ? 1 : 0);
    hi = std::min(hi, top);
    if (lo >= hi) return BTA_OK;
    BTA_CUDA_OK(launch_assemble_seq(c, m == 0 ? BTA_COND : BTA_PRIOR, 0, k.tg(lo), k.tdir, hi - lo, 0,
                                    k.D + (long long)lo * k.d_stride, k.d_stride, st[m][q]));
    return BTA_OK;
  };
  for (int m = 0; m < 2; ++m) {
    const int which = m == 0 ? BTA_COND : BTA_PRIOR;
    BTA_CUDA_OK(cudaEventRecord(ev[12 + m], st[m][0]));           // D, rows, tip of this matrix are assembled
    BTA_CUDA_OK(cudaStreamWaitEvent(st[m][1], ev[12 + m], 0));
    if (!carry) {
      BTA_CUDA_OK(launch_assemble_seq(c, which, 1, 0, 1, ch[m][0].nt, 0, ch[m][0].Bin, bb, st[m][0]));
      BTA_CUDA_OK(launch_assemble_seq(c, which, 1, md.nt - 2, -1, ch[m][1].nt, 1, ch[m][1].Bin, bb, st[m][1]));
    }
  }
  REC(1, st[0][0]);
  REC(5, st[1][0]);

  // ---- forward: four sub-chains, launches interleaved block by block
  for (int m = 0; m < 2; ++m)
    for (int q = 0; q < 2; ++q) BTA_CUDA_OK(chain_forward_begin(ch[m][q], st[m][q]));
  const int maxlen = std::max(ch[0][0].nt, ch[0][1].nt);
  // host staging: one block at a time into the ring slot, once the carry that lived there has been copied out
  auto assemble_slot = [&](int m, int q, int s) -> int {
    const Chain& k = ch[m][q];
    if (s >= k.nt) return BTA_OK;
    BTA_CUDA_OK(cudaStreamWaitEvent(st[m][q], k.ring_ev[s % k.ring], 0));
    BTA_CUDA_OK(launch_assemble_seq(c, m == 0 ? BTA_COND : BTA_PRIOR, 0, k.tg(s), 1, 1, 0, k.Dp(s), 0, st[m][q]));
    return BTA_OK;
  };
  for (int m = 0; m < 2; ++m) {
    if (host)
      BTA_CUDA_OK(launch_assemble_seq(c, m == 0 ? BTA_COND : BTA_PRIOR, 0, h, 1, 1, 0, ch[m][2].D, 0, st[m][0]));
    for (int q = 0; q < 2; ++q) {
      int rc = host ? assemble_slot(m, q, 0) : assemble_range(m, q, 0, 2);
      if (rc != BTA_OK) return rc;
    }
  }
  for (int s = 0; s < maxlen; ++s)
    for (int m = 0; m < 2; ++m)
      for (int q = 0; q < 2; ++q)
        if (s < ch[m][q].nt) {
          if (host) {  // block s+1 receives this step's Schur update
            BTA_CUDA_OK(chain_to_big(ch[m][q], st[m][q]));
            int rc = assemble_slot(m, q, s + 1);
            if (rc != BTA_OK) return rc;
          } else if (s % AHEAD == 0) {  // blocks s+2 .. s+AHEAD+1 (block s+1 receives this step's Schur update)
            BTA_CUDA_OK(chain_to_big(ch[m][q], st[m][q]));
            int rc = assemble_range(m, q, s + 2, s + 2 + AHEAD);
            if (rc != BTA_OK) return rc;
          }
          BTA_CUDA_OK(chain_forward_step(ch[m][q], s, st[m][q]));
        }
  for (int m = 0; m < 2; ++m)
    for (int q = 0; q < 2; ++q) BTA_CUDA_OK(chain_to_big(ch[m][q], st[m][q]));
  for (int m = 0; m < 2; ++m) {
    BTA_CUDA_OK(join_lanes(m, 0));
    BTA_CUDA_OK(join_lanes(m, 1));
    BTA_CUDA_OK(cudaEventRecord(ev[14 + m], st[m][1]));            // down chain eliminated
    BTA_CUDA_OK(cudaStreamWaitEvent(st[m][0], ev[14 + m], 0));
    BTA_CUDA_OK(separator_merge_forward(ch[m][0], ch[m][1], ch[m][2], st[m][0]));
    BTA_CUDA_OK(chain_forward_step(ch[m][2], 0, st[m][0]));
    BTA_CUDA_OK(chain_forward_end(ch[m][2], st[m][0]));
    BTA_CUDA_OK(join_lanes(m, 2));
    BTA_CUDA_OK(launch_logdet_partial(c, m == 0 ? CH_COND : CH_PRIOR, W[m]->dvec, st[m][0]));
  }
  REC(2, st[0][0]);
  REC(6, st[1][0]);

  // ---- backward: separator first, then the two sub-chains outwards
  for (int m = 0; m < 2; ++m) {
    if (value_only && m == 1) break;  // the prior needs no solve
    BTA_CUDA_OK(chain_backward_step(ch[m][2], 0, st[m][0]));
    BTA_CUDA_OK(join_lanes(m, 2));
    BTA_CUDA_OK(cudaEventRecord(ev[16 + m], st[m][0]));
    BTA_CUDA_OK(cudaStreamWaitEvent(st[m][1], ev[16 + m], 0));
  }
  for (int s = maxlen - 1; s >= 0; --s)
    for (int m = 0; m < 2; ++m) {
      if (value_only && m == 1) continue;
      for (int q = 0; q < 2; ++q)
        if (s < ch[m][q].nt) BTA_CUDA_OK(chain_backward_step(ch[m][q], s, st[m][q]));
    }
  // join: everything back onto s0
  for (int m = 0; m < 2; ++m)
    for (int q = 0; q < 2; ++q) {
      BTA_CUDA_OK(join_lanes(m, q));
      if (host) {  // trailing copies of the staging streams
        cudaEvent_t e = c->ev_sw[(c->ev_sw_next++) % BTA_NSW];
        BTA_CUDA_OK(cudaEventRecord(e, ch[m][q].cs));
        BTA_CUDA_OK(cudaStreamWaitEvent(st[m][q], e, 0));
      }
    }
  BTA_CUDA_OK(cudaEventRecord(ev[18], st[0][1]));
  BTA_CUDA_OK(cudaStreamWaitEvent(s0, ev[18], 0));
  BTA_CUDA_OK(cudaMemcpyAsync(wc.x + (long long)md.nt * md.b, ch[0][2].xT, md.a * sizeof(double),
                              cudaMemcpyDeviceToDevice, s0));
  BTA_CUDA_OK(launch_quad_stencil(c, wc.x, s0));
  BTA_CUDA_OK(launch_residual(c, wc.x, s0));
  REC(3, s0);
  BTA_CUDA_OK(cudaEventRecord(ev[19], st[1][1]));
  BTA_CUDA_OK(cudaStreamWaitEvent(st[1][0], ev[19], 0));
  BTA_CUDA_OK(cudaEventRecord(ev[7], st[1][0]));
  BTA_CUDA_OK(cudaStreamWaitEvent(s0, ev[7], 0));

  // ---- scalar assembly (a9)
  REC(10, s0);
  BTA_CUDA_OK(launch_scalars(c, s0));
  const int nout = 1 + md.d + 2 + 3 * md.d + md.k + 1;
  BTA_CUDA_OK(cudaMemcpyAsync(c->host_pinned + 64, c->small + L.out, nout * sizeof(double), cudaMemcpyDeviceToHost,
                              s0));
  BTA_CUDA_OK(cudaMemcpyAsync(c->x_keep, wc.x, md.N * sizeof(double), cudaMemcpyDeviceToDevice, s0));
  REC(8, s0);
  c->have_x = true;
  (void)h;
#undef REC
  return BTA_OK;
}

}  // namespace

namespace {
int value_and_grad_impl(bta_ctx* c, const double* theta, double* f, double* grad, double* stage_ms, void* ws,
                        void* stream, bool value_only) {
  const int gi = value_only ? 1 : 0;
  cudaStream_t s0 = (cudaStream_t)stream;
  const ModelDims& md = c->md;
  DeviceGuard guard(c->device);
  const bool serial = c->opt.serial != 0;
  // Small blocks are launch/latency-bound (tens of thousands of ~2 us kernels): from the second call on, replay
  // the whole gradient as one CUDA graph.  BTA_OPT_GRAPH = 0/1 overrides the size rule (b <= 1024).
  const bool want_graph = c->opt.graph >= 0 ? c->opt.graph == 1 : md.b <= 1024;
  cudaEvent_t* ev = c->ev;
  memcpy(c->host_pinned, theta, md.d * sizeof(double));
  cudaStream_t sync_stream = s0;
  bool timed = true;
  if (want_graph && !serial && c->grad_calls > 0) {
    if (!c->graph_exec[gi] || c->graph_ws[gi] != ws) {
      if (c->graph_exec[gi]) {
        cudaGraphExecDestroy(c->graph_exec[gi]);
        c->graph_exec[gi] = nullptr;
      }
      const long long n0 = c->launches;
      cudaGraph_t graph = nullptr;
      BTA_CUDA_OK(cudaStreamBeginCapture(c->s_main, cudaStreamCaptureModeThreadLocal));
      int rc = use_partitions(c) ? enqueue_gradient_partitioned(c, ws, c->s_main, false, value_only)
               : use_twist(c)    ? enqueue_gradient_twisted(c, ws, c->s_main, false, value_only)
                                 : enqueue_gradient(c, ws, c->s_main, c->s_side, false, value_only);
      cudaError_t ce = cudaStreamEndCapture(c->s_main, &graph);
      if (rc != BTA_OK) return rc;
      BTA_CUDA_OK(ce);
      BTA_CUDA_OK(cudaGraphInstantiate(&c->graph_exec[gi], graph, 0));
      cudaGraphDestroy(graph);
      c->graph_ws[gi] = ws;
      c->graph_launches[gi] = c->launches - n0;
      c->launches = n0;
    }
    BTA_CUDA_OK(cudaEventRecord(ev[11], s0));
    BTA_CUDA_OK(cudaStreamWaitEvent(c->s_main, ev[11], 0));
    BTA_CUDA_OK(cudaEventRecord(ev[0], c->s_main));
    BTA_CUDA_OK(cudaGraphLaunch(c->graph_exec[gi], c->s_main));
    BTA_CUDA_OK(cudaEventRecord(ev[8], c->s_main));
    BTA_CUDA_OK(cudaStreamWaitEvent(s0, ev[8], 0));
    c->launches += c->graph_launches[gi];
    sync_stream = c->s_main;
    timed = false;
  } else {
    int rc;
    if (use_partitions(c)) {
      BTA_CUDA_OK(cudaEventRecord(ev[11], s0));
      BTA_CUDA_OK(cudaStreamWaitEvent(c->s_main, ev[11], 0));
      rc = enqueue_gradient_partitioned(c, ws, c->s_main, true, value_only);
      if (rc != BTA_OK) return rc;
      BTA_CUDA_OK(cudaEventRecord(ev[20], c->s_main));
      BTA_CUDA_OK(cudaStreamWaitEvent(s0, ev[20], 0));
      sync_stream = c->s_main;
      timed = false;  // only the total is timed in this mode
    } else if (use_twist(c) && !serial) {
      // run on the library's own prioritised streams; the caller's stream only orders the call
      BTA_CUDA_OK(cudaEventRecord(ev[11], s0));
      BTA_CUDA_OK(cudaStreamWaitEvent(c->s_main, ev[11], 0));
      rc = enqueue_gradient_twisted(c, ws, c->s_main, true, value_only);
      if (rc != BTA_OK) return rc;
      BTA_CUDA_OK(cudaEventRecord(ev[20], c->s_main));
      BTA_CUDA_OK(cudaStreamWaitEvent(s0, ev[20], 0));
      sync_stream = c->s_main;
    } else {
      rc = enqueue_gradient(c, ws, s0, serial ? s0 : c->s_side, true, value_only);
      if (rc != BTA_OK) return rc;
    }
  }
  c->grad_calls++;
  int rc = check_pivot(c, sync_stream);
  if (c->trace_on && !c->trace.empty()) {  // diagnostic timeline: "<chain> <t> <tag> <ms since the call started>"
    if (FILE* fp = fopen(getenv("BTA_TRACE"), "w")) {
      for (auto& r : c->trace) {
        float ms = 0.f;
        cudaEventSynchronize(r.e);
        cudaEventElapsedTime(&ms, ev[0], r.e);
        fprintf(fp, "%d %d %d %.4f\n", r.chain, r.t, r.tag, ms);
      }
      fclose(fp);
    }
    for (auto& r : c->trace) cudaEventDestroy(r.e);
    c->trace.clear();
  }  // synchronises the stream (and, through ev[7], the side stream)
  const double* o = c->host_pinned + 64;
  if (f) *f = o[0];
  if (grad && !value_only) memcpy(grad, o + 1, md.d * sizeof(double));
  c->last_ld[0] = o[1 + md.d];
  c->last_ld[1] = o[1 + md.d + 1];
  c->last_parts.assign(o + 1 + md.d + 2, o + 1 + md.d + 2 + 3 * md.d);
  c->last_rss.assign(o + 1 + md.d + 2 + 3 * md.d, o + 1 + md.d + 2 + 3 * md.d + md.k);
  c->last_quad = o[1 + md.d + 2 + 3 * md.d + md.k];
  if (stage_ms && !timed) {
    for (int i = 0; i < BTA_NSTAGES; ++i) stage_ms[i] = 0.0;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, ev[0], ev[8]);
    stage_ms[BTA_STAGE_TOTAL] = ms;
  } else if (stage_ms) {
    auto el = [&](int a_, int b_) {
      float ms = 0.f;
      cudaEventElapsedTime(&ms, ev[a_], ev[b_]);
      return (double)ms;
    };
    stage_ms[BTA_STAGE_ASSEMBLE] = el(9, 1) + el(4, 5);
    stage_ms[BTA_STAGE_FWD_QC] = el(1, 2);
    stage_ms[BTA_STAGE_BWD_QC] = el(2, 3);
    stage_ms[BTA_STAGE_FWD_QP] = el(5, 6);
    stage_ms[BTA_STAGE_BWD_QP] = el(6, 7);
    stage_ms[BTA_STAGE_SCALARS] = el(10, 8);
    stage_ms[BTA_STAGE_TOTAL] = el(0, 8);
  }
  return rc;
}
}  // namespace

extern "C" int inla_value_and_grad(bta_ctx* c, const double* theta, double* f, double* grad, double* stage_ms,
                                   void* ws, void* stream) {
  if (!c || !theta || !ws) return bad("inla_value_and_grad: null ctx, theta or workspace");
  return value_and_grad_impl(c, theta, f, grad, stage_ms, ws, stream, false);
}

extern "C" int inla_value(bta_ctx* c, const double* theta, double* f, void* ws, void* stream) {
  if (!c || !theta || !ws) return bad("inla_value: null ctx, theta or workspace");
  return value_and_grad_impl(c, theta, f, nullptr, nullptr, ws, stream, true);
}

extern "C" int inla_fd_grad(bta_ctx* c, const double* theta, double h, double* f, double* grad, void* ws,
                            void* stream) {
  if (!c || !theta || !ws || !grad) return bad("inla_fd_grad: null ctx, theta, grad or workspace");
  if (!(h > 0.0)) return bad("inla_fd_grad: h must be positive");
  const int d = c->md.d;
  std::vector<double> th(theta, theta + d);
  double f0 = 0.0;
  int rc = value_and_grad_impl(c, th.data(), &f0, nullptr, nullptr, ws, stream, true);
  if (rc != BTA_OK) return rc;
  if (f) *f = f0;
  for (int j = 0; j < d; ++j) {
    double fp = 0.0, fm = 0.0;
    th[j] = theta[j] + h;
    if ((rc = value_and_grad_impl(c, th.data(), &fp, nullptr, nullptr, ws, stream, true)) != BTA_OK) return rc;
    th[j] = theta[j] - h;
    if ((rc = value_and_grad_impl(c, th.data(), &fm, nullptr, nullptr, ws, stream, true)) != BTA_OK) return rc;
    th[j] = theta[j];
    grad[j] = (fp - fm) / (2.0 * h);
  }
  return BTA_OK;
}

extern "C" int inla_hessian(bta_ctx* c, const double* theta, double h, double* f, double* grad, double* H, void* ws,
                            void* stream) {
  if (!c || !theta || !ws || !H) return bad("inla_hessian: null ctx, theta, H or workspace");
  if (!(h > 0.0)) return bad("inla_hessian: h must be positive");
  const int d = c->md.d;
  std::vector<double> th(theta, theta + d), gp(d), gm(d), g0(d);
  double f0 = 0.0;
  int rc = value_and_grad_impl(c, th.data(), &f0, g0.data(), nullptr, ws, stream, false);
  if (rc != BTA_OK) return rc;
  if (f) *f = f0;
  if (grad) memcpy(grad, g0.data(), d * sizeof(double));
  for (int j = 0; j < d; ++j) {
    th[j] = theta[j] + h;
    if ((rc = value_and_grad_impl(c, th.data(), nullptr, gp.data(), nullptr, ws, stream, false)) != BTA_OK) return rc;
    th[j] = theta[j] - h;
    if ((rc = value_and_grad_impl(c, th.data(), nullptr, gm.data(), nullptr, ws, stream, false)) != BTA_OK) return rc;
    th[j] = theta[j];
    for (int i = 0; i < d; ++i) H[i * d + j] = (gp[i] - gm[i]) / (2.0 * h);
  }
  return BTA_OK;
}

extern "C" int inla_optimize(bta_ctx* c, const double* theta0, int max_iter, double gtol, double* theta_opt,
                             double* f_opt, double* grad_opt, int* iters, int* evals, void* ws, void* stream) {
  if (!c || !theta0 || !ws) return bad("inla_optimize: null ctx, theta0 or workspace");
  if (max_iter < 0 || !(gtol >= 0.0)) return bad("inla_optimize: max_iter >= 0 and gtol >= 0 required");
  const int d = c->md.d, mem = 10;
  // minimise phi = -f;  g = -grad f
  std::vector<double> x(theta0, theta0 + d), g(d), xn(d), gn(d), dir(d), q(d);
  std::vector<std::vector<double>> S, Y;
  std::vector<double> rho;
  double phi = 0.0;
  int nev = 0, it = 0;
  auto eval = [&](const std::vector<double>& th, double& ph, std::vector<double>& gr) -> int {
    double fv = 0.0;
    int rc = value_and_grad_impl(c, th.data(), &fv, gr.data(), nullptr, ws, stream, false);
    ++nev;
    ph = -fv;
    for (int i = 0; i < d; ++i) gr[i] = -gr[i];
    return rc;
  };
  auto dot = [&](const std::vector<double>& a_, const std::vector<double>& b_) {
    double s_ = 0.0;
    for (int i = 0; i < d; ++i) s_ += a_[i] * b_[i];
    return s_;
  };
  int rc = eval(x, phi, g);
  if (rc != BTA_OK) return rc;
  for (; it < max_iter; ++it) {
    double gmax = 0.0;
    for (int i = 0; i < d; ++i) gmax = std::max(gmax, std::fabs(g[i]));
    if (gmax <= gtol) break;
    // two-loop recursion
    q = g;
    const int mcur = (int)S.size();
    std::vector<double> al(mcur);
    for (int i = mcur - 1; i >= 0; --i) {
      al[i] = rho[i] * dot(S[i], q);
      for (int j = 0; j < d; ++j) q[j] -= al[i] * Y[i][j];
    }
    double gamma = 1.0;
    if (mcur > 0) gamma = dot(S[mcur - 1], Y[mcur - 1]) / dot(Y[mcur - 1], Y[mcur - 1]);
    for (int j = 0; j < d; ++j) q[j] *= gamma;
    for (int i = 0; i < mcur; ++i) {
      const double be = rho[i] * dot(Y[i], q);
      for (int j = 0; j < d; ++j) q[j] += (al[i] - be) * S[i][j];
    }
    for (int j = 0; j < d; ++j) dir[j] = -q[j];
    double slope = dot(g, dir);
    if (!(slope < 0.0)) {  // not a descent direction: restart from steepest descent
      S.clear();
      Y.clear();
      rho.clear();
      for (int j = 0; j < d; ++j) dir[j] = -g[j];
      slope = dot(g, dir);
    }
    double step = (mcur == 0) ? std::min(1.0, 1.0 / std::max(gmax, 1e-300)) : 1.0;
    double phin = 0.0;
    bool ok = false;
    for (int ls = 0; ls < 30; ++ls) {
      for (int j = 0; j < d; ++j) xn[j] = x[j] + step * dir[j];
      rc = eval(xn, phin, gn);
      if (rc == BTA_OK && std::isfinite(phin) && phin <= phi + 1e-4 * step * slope) {
        ok = true;
        break;
      }
      if (rc != BTA_OK && rc != BTA_ERR_NOTSPD) return rc;
      step *= 0.5;
    }
    if (!ok) break;  // no progress possible at this precision
    std::vector<double> sv(d), yv(d);
    for (int j = 0; j < d; ++j) {
      sv[j] = xn[j] - x[j];
      yv[j] = gn[j] - g[j];
    }
    const double sy = dot(sv, yv);
    if (sy > 1e-12 * std::sqrt(dot(sv, sv) * dot(yv, yv))) {
      S.push_back(sv);
      Y.push_back(yv);
      rho.push_back(1.0 / sy);
      if ((int)S.size() > mem) {
        S.erase(S.begin());
        Y.erase(Y.begin());
        rho.erase(rho.begin());
      }
    }
    x = xn;
    g = gn;
    phi = phin;
  }
  if (theta_opt) memcpy(theta_opt, x.data(), d * sizeof(double));
  if (f_opt) *f_opt = -phi;
  if (grad_opt)
    for (int i = 0; i < d; ++i) grad_opt[i] = -g[i];
  if (iters) *iters = it;
  if (evals) *evals = nev;
  return BTA_OK;
}

extern "C" int bta_last_intermediates(bta_ctx* c, double* ld, double* x, double* parts, double* rss, double* quad,
                                      double* ZT) {
  if (!c) return bad("bta_last_intermediates: null ctx");
  DeviceGuard guard(c->device);
  if (ld) {
    ld[0] = c->last_ld[0];
    ld[1] = c->last_ld[1];
  }
  if (parts && !c->last_parts.empty()) memcpy(parts, c->last_parts.data(), c->last_parts.size() * sizeof(double));
  if (rss && !c->last_rss.empty()) memcpy(rss, c->last_rss.data(), c->last_rss.size() * sizeof(double));
  if (quad) *quad = c->last_quad;
  if (ZT) {
    SmallLayout L = small_layout(c->md);
    BTA_CUDA_OK(cudaMemcpy(ZT, c->small + L.ZT[CH_COND], sizeof(double) * c->md.a * c->md.a, cudaMemcpyDeviceToHost));
  }
  if (x) {
    if (!c->have_x) return bad("bta_last_intermediates: no gradient has been computed yet");
    BTA_CUDA_OK(cudaMemcpy(x, c->x_keep, c->md.N * sizeof(double), cudaMemcpyDeviceToHost));
  }
  return BTA_OK;
}

extern "C" size_t bta_workspace_bytes(const bta_ctx* c) {
  if (!c) return 0;
  const size_t one = grad_ws_bytes(c->md, c->store_mode);
  const size_t two = c->md.nt >= 3 ? twist_ws_bytes(c->md, c->store_mode) : (size_t)0;
  if (use_partitions(c)) return part_ws_bytes(c);
  if (c->store_mode == BTA_STORE_HOST && use_twist(c)) return two;  // O(b^2): the point of the mode
  return one > two ? one : two;
}
