// Time-domain partitioning with P partitions and a reduced system (§III-C a-b; SURVEY.md §8(f)
// NEXT-3), inside one GPU and -- through the phase calls of include/bta.h -- across ranks.
//
// The nt time blocks are cut into P contiguous partitions [s_p, e_p].  Partition 0 is eliminated downwards and ends at
// its boundary block e_0; a partition p >= 1 has two boundary blocks (s_p, e_p): its interior blocks s_p+1 .. e_p-1 are
// eliminated downwards with a fill coupling to s_p (sweep.h: Fill).  The 2P-1 boundary blocks, in the order
// e_0, s_1, e_1, ..., s_{P-1}, e_{P-1}, form a reduced BTA system (sub-diagonal blocks: the original B_{e_p} between
// e_p and s_{p+1}, the fill block Q~[e_p, s_p] between s_p and e_p) that is factored and selectively inverted by the
// ordinary chain code; its Sigma blocks then seed the backward sweeps of the interiors (reverse order).
//   Phase 1  (no communication): interior chains of all partitions concurrently, one stream each
//   Phase 2  : reduced system -- forward, tip, backward with selected inversion and the traces of the boundary blocks
//   Phase 1' : interior backward sweeps concurrently
// With ranks (bta_part_*): a rank runs Phase 1 / 1' for its own partition only; the boundary blocks, fill blocks, their
// stack rows and the tip contributions are exchanged once (all-gather), every rank solves the reduced system, and
// the per-block partial sums are summed once (all-reduce) -- the paper's communication pattern.
// Factor mode only (the carries of the interiors are not staged).  Costs ~2.7x the flops per interior block of a
// partition p >= 1: it buys concurrency (latency-bound models) and the multi-rank form, not single-GPU throughput.
#include <algorithm>
#include <cstring>

#include "api_util.h"

namespace {

struct Plan {
  int P = 0, nred = 0;
  int s[BTA_PMAX], e[BTA_PMAX];
  int first_int(int p) const { return p == 0 ? 0 : s[p] + 1; }          // first interior block
  int nint(int p) const { return e[p] - first_int(p); }                 // interior blocks (eliminated in Phase 1)
  int q_s(int p) const { return 2 * p - 1; }                            // reduced index of s_p (p >= 1)
  int q_e(int p) const { return 2 * p; }                                // reduced index of e_p
};

// Partition sizes: an interior block of a partition p >= 1 costs ~2.7x one of partition 0 (fill), so partition 0 is
// made ~2.7x longer; every partition p >= 1 needs its two boundary blocks.
Plan make_plan(int nt, int want) {
  Plan pl;
  int P = std::max(2, std::min(want, BTA_PMAX));
  while (P > 2 && nt < 2 * P - 1) --P;
  int np = (int)((nt + 5.4) / (2.7 + P - 1) + 0.5);
  np = std::max(2, np);
  while (np > 2 && nt - (P - 1) * np < 1) --np;
  const int n0 = nt - (P - 1) * np;
  pl.P = P;
  pl.nred = 2 * P - 1;
  pl.s[0] = 0;
  pl.e[0] = n0 - 1;
  for (int p = 1; p < P; ++p) {
    pl.s[p] = pl.e[p - 1] + 1;
    pl.e[p] = pl.s[p] + np - 1;
  }
  return pl;
}

struct SubWs {
  double *W1, *W2, *W3, *H, *Ftil, *ubuf, *Ebuf, *Ybuf, *ZC0, *ZC1, *part, *Tt, *B;
};
struct PartWs {
  double *D, *LF, *dvec, *T, *Rin, *Rout, *x, *rtip;
  double *BredIn, *BredOut, *RinRed, *RoutRed, *ZCred;
  SubWs sub[BTA_PMAX + 1];  // [P] = the reduced chain
};

PartWs carve_part(Bump& bp, const ModelDims& md, const Plan& pl, bool cond) {
  PartWs w{};
  const size_t bb = (size_t)md.b * md.b;
  const int PR = md.a + 1;
  const size_t rs = (size_t)PR * md.b;
  w.D = bp.take(bb * md.nt);
  w.LF = bp.take(bb * md.nt);
  w.dvec = bp.take(md.N);
  w.T = bp.take(md.a * md.a);
  w.BredIn = bp.take(bb * pl.nred);
  w.BredOut = bp.take(bb * pl.nred);
  if (cond) {
    w.Rin = bp.take((size_t)md.nt * rs);
    w.Rout = bp.take((size_t)md.nt * rs);
    w.x = bp.take(md.N);
    w.rtip = bp.take(md.a);
    w.RinRed = bp.take(rs * pl.nred);
    w.RoutRed = bp.take(rs * pl.nred);
    w.ZCred = bp.take((size_t)md.a * md.b * pl.nred);
  }
  for (int p = 0; p <= pl.P; ++p) {
    SubWs& s = w.sub[p];
    s.W1 = bp.take(bb);
    s.W2 = bp.take(bb);
    s.W3 = bp.take(bb);
    s.Tt = bp.take(md.a * (md.a + 1));
    if (p < pl.P) {
      s.B = bp.take(bb * (pl.nint(p) + 1));
      if (p > 0) {
        s.H = bp.take(bb);
        s.Ftil = bp.take(bb);
      }
    }
    if (cond) {
      s.ubuf = bp.take(md.b);
      s.Ebuf = bp.take((size_t)md.a * md.b);
      s.Ybuf = bp.take((size_t)md.a * md.b);
      s.ZC0 = bp.take((size_t)md.a * md.b);
      s.ZC1 = bp.take((size_t)md.a * md.b);
      s.part = bp.take(skinny_nn_part_doubles(PR, md.b, md.b));
    }
  }
  return w;
}

__global__ void vec_add_kernel(int n, const double* __restrict__ src, double* __restrict__ dst) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) dst[i] += src[i];
}

#define CKP(call)                                          \
  do {                                                     \
    cudaError_t e_ = (call);                               \
    if (e_ != cudaSuccess) {                               \
      bta_set_error_cuda(e_, #call, __FILE__, __LINE__);   \
      return BTA_ERR_CUDA;                                 \
    }                                                      \
  } while (0)

int ensure_streams(bta_ctx* c, int P) {
  int lo = 0, hi = 0;
  CKP(cudaDeviceGetStreamPriorityRange(&lo, &hi));
  for (int m = 0; m < 2; ++m)
    for (int p = 0; p < P; ++p) {
      if (!c->s_part[m][p]) CKP(cudaStreamCreateWithPriority(&c->s_part[m][p], cudaStreamNonBlocking, lo));
      if (!c->s_part_hi[m][p]) CKP(cudaStreamCreateWithPriority(&c->s_part_hi[m][p], cudaStreamNonBlocking, hi));
      if (!c->s_part_x[m][p]) CKP(cudaStreamCreateWithPriority(&c->s_part_x[m][p], cudaStreamNonBlocking, lo));
      if (!c->s_part_r[m][p]) CKP(cudaStreamCreateWithPriority(&c->s_part_r[m][p], cudaStreamNonBlocking, hi));
    }
  return BTA_OK;
}

}  // namespace

bool use_partitions(const bta_ctx* c) {
  return c->opt.partitions >= 2 && c->md.nt >= 3 && c->store_mode == BTA_STORE_FACTOR && !c->opt.serial;
}

extern "C" int bta_partition_plan(const bta_ctx* c, int partitions, int32_t* first, int32_t* last) {
  if (!c) return 0;
  const Plan pl = make_plan(c->md.nt, partitions);
  for (int p = 0; p < pl.P; ++p) {
    if (first) first[p] = pl.s[p];
    if (last) last[p] = pl.e[p];
  }
  return pl.P;
}

// ------------------------------------------------------------------------------------------------
// One gradient with P partitions per matrix, in stages.  nranks == 1: all partitions are local (one GPU).  nranks > 1:
// rank r owns partition r; the stages map onto the paper's phases:
//   phase1  = assembly + Phase 1 of the local partitions + merge into their boundary blocks (+ pack the slab)
//   phase2  = (unpack all slabs +) reduced system forward / backward + Phase 1' of the local partitions + the local
//             per-block partial sums
//   finish  = scalar assembly from the (summed) partial sums
// All work is forked from and joined back into s0 (so a single-rank call can be captured into a CUDA graph).
// ------------------------------------------------------------------------------------------------
namespace {

__global__ void fill_kernel(long long n, double v, double* __restrict__ dst) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) dst[i] = v;
}

struct PartRun {
  bta_ctx* c = nullptr;
  Plan pl;
  PartWs W[2];
  Chain pc[2][BTA_PMAX], red[2];
  Fill fills[2][BTA_PMAX];
  int tmap[2 * BTA_PMAX], bmap[2 * BTA_PMAX];
  double* dmap[2][2 * BTA_PMAX];
  cudaStream_t S[2][BTA_PMAX];
  cudaStream_t s0 = nullptr;
  SmallLayout L;
  bool value_only = false;
  int rank = 0, nranks = 1;
  double* dvec_dummy = nullptr;   // ranks != 0: where the (redundant) reduced chain puts its diag(L)
  long long bb = 0, rs = 0;
  int b = 0, a = 0, PR = 0;

  bool local(int p) const { return nranks == 1 || p == rank; }
  cudaError_t link(cudaStream_t from, cudaStream_t to) {
    if (from == to) return cudaSuccess;
    cudaEvent_t e = c->ev_sw[(c->ev_sw_next++) % BTA_NSW];
    cudaError_t ce = cudaEventRecord(e, from);
    return ce != cudaSuccess ? ce : cudaStreamWaitEvent(to, e, 0);
  }
  size_t slab_doubles() const { return 2 * (3 * (size_t)bb + (size_t)a * (a + 1)) + 2 * (size_t)rs; }

  int init(bta_ctx* ctx, void* ws, cudaStream_t stream, bool vonly, int rank_, int nranks_);
  int phase1();
  int pack(double* slab);
  int unpack(const double* gathered);
  int phase2();
  int finish(bool timed);
};

int PartRun::init(bta_ctx* ctx, void* ws, cudaStream_t stream, bool vonly, int rank_, int nranks_) {
  c = ctx;
  s0 = stream;
  value_only = vonly;
  rank = rank_;
  nranks = nranks_;
  const ModelDims& md = c->md;
  pl = make_plan(md.nt, nranks > 1 ? nranks : c->opt.partitions);
  if (nranks > 1 && pl.P != nranks) return bad("inla_part_*: nt is too small for that many ranks (need nt >= 2 nranks - 1)");
  const int P = pl.P, nred = pl.nred;
  if (int rc = ensure_streams(c, P); rc != BTA_OK) return rc;
  Bump bp(ws);
  W[0] = carve_part(bp, md, pl, true);
  W[1] = carve_part(bp, md, pl, false);
  dvec_dummy = bp.take(md.N);
  L = small_layout(md);
  bb = (long long)md.b * md.b;
  b = md.b;
  a = md.a;
  PR = a + 1;
  rs = (long long)PR * b;
  // streams: [matrix][partition]; (0, 0) is the caller-ordered stream s0; the reduced chains run on [m][0]
  for (int m = 0; m < 2; ++m)
    for (int p = 0; p < P; ++p) S[m][p] = (m == 0 && p == 0) ? s0 : c->s_part[m][p];
  // host tables of the reduced system (same for both matrices but for the block pointers)
  tmap[0] = pl.e[0];
  for (int p = 1; p < P; ++p) {
    tmap[pl.q_s(p)] = pl.s[p];
    tmap[pl.q_e(p)] = pl.e[p];
  }
  for (int q = 0; q < nred - 1; ++q) {
    if (q % 2 == 0)
      bmap[q] = tmap[q];                                        // e_p -> s_{p+1}: the original B_{e_p}
    else
      bmap[q] = pl.nint((q + 1) / 2) == 0 ? tmap[q] : -1;       // s_p -> e_p: B_{s_p} if adjacent, else a fill block
  }
  bmap[nred - 1] = -1;
  for (int m = 0; m < 2; ++m)
    for (int q = 0; q < nred; ++q) dmap[m][q] = W[m].D + (long long)tmap[q] * bb;

  for (int m = 0; m < 2; ++m) {
    const bool cond = m == 0;
    const int chs = cond ? CH_COND : CH_PRIOR;
    const PartWs& w = W[m];
    for (int p = 0; p <= P; ++p) {
      Chain& k = p < P ? pc[m][p] : red[m];
      const SubWs& s = w.sub[p];
      k = Chain();
      k.c = c;
      k.chain = chs;
      k.which = cond ? BTA_COND : BTA_PRIOR;
      k.b = b;
      k.a = a;
      k.nr = cond ? 1 : 0;
      k.arrow_rows = cond;
      k.selinv = k.contract = !value_only;
      k.b_stride = bb;
      k.T = w.T;
      k.ldT = a;
      k.W1 = s.W1;
      k.W2 = s.W2;
      k.W3 = s.W3;
      k.dvec = w.dvec;
      k.LT = c->small + L.LT[chs];
      k.zT = c->small + L.zT[chs];
      k.xT = c->small + L.xT[chs];
      k.ZT = c->small + L.ZT[chs];
      if (cond) {
        k.rhs_tip = w.rtip;
        k.rhs_tip_stride = a;
        k.ubuf = s.ubuf;
        k.Ebuf = s.Ebuf;
        k.Ybuf = s.Ybuf;
        k.ZC[0] = s.ZC0;
        k.ZC[1] = s.ZC1;
        k.part = s.part;
        k.xout = w.x;
        k.ld_x = md.N;
      }
      const int sp = m * (BTA_PMAX + 1) + p;  // slot of this chain's events
      if (c->opt.lanes) k.hi = p < P ? c->s_part_hi[m][p] : c->s_part_hi[m][0];
      k.lanes_bwd = c->opt.lanes != 2;
      if (c->opt.split) k.xs = p < P ? c->s_part_x[m][p] : c->s_part_x[m][0];
      k.pipe_ev = c->ev_pipe[sp];
      if (c->opt.rows && b <= 1024) k.rs = p < P ? c->s_part_r[m][p] : c->s_part_r[m][0];
      if (p < P) {  // interior chain of partition p
        const int i0 = pl.first_int(p);
        k.nt = pl.nint(p);
        k.t0 = i0;
        k.tdir = 1;
        k.tail_coupling = true;
        k.tt_zero = p > 0;
        k.D = w.D + (long long)i0 * bb;
        k.d_stride = bb;
        k.Bin = s.B + bb;   // B_t assembled into slot t+1, L_Bt written to slot t
        k.Bout = s.B;
        k.Tt = (p == 0 && nranks == 1) ? c->small + L.Tt[chs] : s.Tt;
        if (cond) {
          k.Rin = w.Rin + (long long)i0 * rs;
          k.Rout = w.Rout + (long long)i0 * rs;
          k.rin_stride = k.rout_stride = rs;
          k.ld_rin = k.ld_rout = b;
        }
        // what the last interior block sees as its "next" block: the boundary e_p of the reduced system
        k.sep_x = cond ? w.x + (long long)pl.e[p] * b : nullptr;
        k.sep_ZD = w.D + (long long)pl.e[p] * bb;                                    // Sigma[e,e], written in place
        k.sep_ZC = cond ? w.ZCred + (long long)pl.q_e(p) * a * b : nullptr;
        if (p > 0) {
          Fill& f = fills[m][p];
          f = Fill();
          f.LF = w.LF + (long long)i0 * bb;
          f.lf_stride = bb;
          f.Ftil = s.Ftil;
          f.H = s.H;
          f.Ds = w.D + (long long)pl.s[p] * bb;
          f.Rs = cond ? w.RinRed + (long long)pl.q_s(p) * rs : nullptr;
          f.ld_rs = b;
          f.Bse = w.BredIn + (long long)pl.q_s(p) * bb;
          f.ZDs = w.D + (long long)pl.s[p] * bb;
          f.ZCs = cond ? w.ZCred + (long long)pl.q_s(p) * a * b : nullptr;
          f.xs = cond ? w.x + (long long)pl.s[p] * b : nullptr;
          f.ld_xs = md.N;
          f.ZFe = w.BredOut + (long long)pl.q_s(p) * bb;                             // Sigma[e_p, s_p] (reduced Z_B)
          f.tb_first = pl.s[p];
          k.fill = &f;
        }
      } else {  // the reduced chain
        k.nt = nred;
        k.tmap = tmap;
        k.bmap = bmap;
        k.dmap = dmap[m];
        k.D = w.D;
        k.d_stride = bb;
        k.Bin = w.BredIn;
        k.Bout = w.BredOut;
        k.Tt = c->small + L.Tt[chs];
        k.selinv_inplace = !value_only;   // Sigma of the boundary blocks stays in their slots for Phase 1'
        if (nranks > 1 && rank != 0) {    // every rank solves the reduced system; rank 0 alone counts it
          k.contract = false;
          k.dvec = dvec_dummy;
        }
        if (cond) {
          k.Rin = w.RinRed;
          k.Rout = w.RoutRed;
          k.rin_stride = k.rout_stride = rs;
          k.ld_rin = k.ld_rout = b;
          k.Cout = w.ZCred;
          k.cout_stride = (long long)a * b;
        }
      }
    }
  }
  return BTA_OK;
}

int PartRun::phase1() {
  const ModelDims& md = c->md;
  const int P = pl.P;
  CKP(cudaMemcpyAsync(c->theta_dev, c->host_pinned, md.d * sizeof(double), cudaMemcpyHostToDevice, s0));
  CKP(launch_theta_prep(c, s0));
  CKP(cudaMemsetAsync(c->pivot_flag, 0xFF, sizeof(unsigned long long), s0));
  if (nranks > 1) {  // partial sums of blocks this rank does not own stay zero; diag(L) entries it does not own stay 1
    CKP(cudaMemsetAsync(c->small, 0, L.Tt[0] * sizeof(double), s0));
    for (int m = 0; m < 2; ++m) {
      fill_kernel<<<(unsigned)((md.N + 255) / 256), 256, 0, s0>>>(md.N, 1.0, W[m].dvec);
      BTA_COUNT(c);
    }
  }
  // stack rows of all blocks, tips
  CKP(launch_assemble(c, BTA_COND, nullptr, bb, nullptr, 0, W[0].Rin, rs, W[0].T, a, W[0].Rin + (long long)a * b, rs,
                      W[0].rtip, 1, s0));
  for (int m = 0; m < 2; ++m)
    for (int p = 0; p < P; ++p) CKP(link(s0, S[m][p]));
  CKP(launch_assemble(c, BTA_PRIOR, nullptr, bb, nullptr, 0, nullptr, 0, W[1].T, a, nullptr, 0, nullptr, 0, S[1][0]));

  // ---- assembly per local partition: its diagonal blocks (boundaries included), interior couplings, fill seed, and
  //      the stack rows of its boundary blocks; the reduced system's original couplings B_{e_p} (every rank, all p)
  for (int m = 0; m < 2; ++m) {
    const int which = m == 0 ? BTA_COND : BTA_PRIOR;
    const PartWs& w = W[m];
    for (int p = 0; p < P; ++p) {
      cudaStream_t st = S[m][p];
      if (p < P - 1) CKP(launch_assemble_block(c, which, 1, pl.e[p], 0, w.BredIn + (long long)pl.q_e(p) * bb, st));
      if (!local(p)) continue;
      const int i0 = pl.first_int(p), ni = pl.nint(p);
      CKP(launch_assemble_seq(c, which, 0, pl.s[p], 1, pl.e[p] - pl.s[p] + 1, 0, w.D + (long long)pl.s[p] * bb, bb, st));
      if (ni > 0) CKP(launch_assemble_seq(c, which, 1, i0, 1, ni, 0, pc[m][p].Bin, bb, st));
      if (p > 0) {
        if (ni > 0)
          CKP(launch_assemble_block(c, which, 1, pl.s[p], 1, w.sub[p].Ftil, st));                 // F~_{s+1} = B_s^T
        else
          CKP(launch_assemble_block(c, which, 1, pl.s[p], 0, w.BredIn + (long long)pl.q_s(p) * bb, st));
      }
      if (m == 0) {
        if (p > 0)
          CKP(cudaMemcpyAsync(w.RinRed + (long long)pl.q_s(p) * rs, w.Rin + (long long)pl.s[p] * rs, rs * sizeof(double),
                              cudaMemcpyDeviceToDevice, st));
        CKP(cudaMemcpyAsync(w.RinRed + (long long)pl.q_e(p) * rs, w.Rin + (long long)pl.e[p] * rs, rs * sizeof(double),
                            cudaMemcpyDeviceToDevice, st));
      }
    }
  }

  // ---- Phase 1: the interior chains of the local partitions, launches interleaved block by block
  int maxlen = 0;
  for (int p = 0; p < P; ++p)
    if (local(p)) maxlen = std::max(maxlen, pl.nint(p));
  for (int m = 0; m < 2; ++m)
    for (int p = 0; p < P; ++p)
      if (local(p)) CKP(chain_forward_begin(pc[m][p], S[m][p]));
  for (int s = 0; s < maxlen; ++s)
    for (int m = 0; m < 2; ++m)
      for (int p = 0; p < P; ++p)
        if (local(p) && s < pc[m][p].nt) CKP(chain_forward_step(pc[m][p], s, S[m][p]));
  // merge into the reduced system: Schur update and stack update of e_p from the last interior block, tip sums
  for (int m = 0; m < 2; ++m) {
    const PartWs& w = W[m];
    for (int p = 0; p < P; ++p) {
      if (!local(p)) continue;
      Chain& k = pc[m][p];
      cudaStream_t st = S[m][p];
      CKP(chain_to_big(k, st));
      if (k.nt > 0) {
        const double* LB = k.Bout + (long long)(k.nt - 1) * bb;
        if (m == 0) {
          double* Re = w.RinRed + (long long)pl.q_e(p) * rs;
          CKP(launch_skinny_nt(PR, b, b, k.Rout + (long long)(k.nt - 1) * rs, b, LB, b, 0, -1.0, 1.0, Re, b, Re, b, st));
          BTA_COUNT(c);
        }
        GemmArgs g{LB, LB, w.D + (long long)pl.e[p] * bb, b, b, b, b, b, b, -1.0, 1.0, GEMM_NT, KLO_ZERO, KHI_K, OUT_LOWER,
                   nullptr, 0, 0};
        CKP(launch_gemm(g, st));
        BTA_COUNT(c);
      }
      if (nranks == 1 && p > 0) {
        CKP(link(st, S[m][0]));
        if (a > 0) {
          const int n = a * (a + red[m].nr);
          vec_add_kernel<<<(n + 127) / 128, 128, 0, S[m][0]>>>(n, k.Tt, red[m].Tt);
          BTA_COUNT(c);
        }
      }
    }
  }
  return BTA_OK;
}

// Slab of the local partition p = rank, per matrix m: [D~(s_p) | D~(e_p) | Q~(e_p, s_p) | tip accumulator], and for
// Q_c the stack rows [C~; r~] of s_p and e_p.  Partition 0 leaves the s_p and fill parts unused (uniform slab size).
int PartRun::pack(double* slab) {
  const int p = rank;
  size_t off = 0;
  for (int m = 0; m < 2; ++m) {
    const PartWs& w = W[m];
    cudaStream_t st = S[m][p];
    auto put = [&](const double* src, size_t n) -> cudaError_t {
      cudaError_t e = src ? cudaMemcpyAsync(slab + off, src, n * sizeof(double), cudaMemcpyDeviceToDevice, st) : cudaSuccess;
      off += n;
      return e;
    };
    CKP(put(p > 0 ? w.D + (long long)pl.s[p] * bb : nullptr, bb));
    CKP(put(w.D + (long long)pl.e[p] * bb, bb));
    CKP(put(p > 0 ? w.BredIn + (long long)pl.q_s(p) * bb : nullptr, bb));
    CKP(put(pc[m][p].Tt, (size_t)a * (a + 1)));
    if (m == 0) {
      CKP(put(p > 0 ? w.RinRed + (long long)pl.q_s(p) * rs : nullptr, rs));
      CKP(put(w.RinRed + (long long)pl.q_e(p) * rs, rs));
    }
    CKP(link(st, s0));
  }
  return BTA_OK;
}

int PartRun::unpack(const double* gathered) {
  const size_t sd = slab_doubles();
  for (int m = 0; m < 2; ++m) {
    const PartWs& w = W[m];
    cudaStream_t st = S[m][0];
    CKP(link(s0, st));
    const int ntip = a * (a + red[m].nr);
    if (ntip > 0) CKP(cudaMemsetAsync(red[m].Tt, 0, ntip * sizeof(double), st));
    for (int p = 0; p < pl.P; ++p) {
      const double* src = gathered + (size_t)p * sd + (m == 0 ? 0 : 3 * (size_t)bb + (size_t)a * (a + 1) + 2 * (size_t)rs);
      auto get = [&](double* dst, size_t n) -> cudaError_t {
        cudaError_t e = dst ? cudaMemcpyAsync(dst, src, n * sizeof(double), cudaMemcpyDeviceToDevice, st) : cudaSuccess;
        src += n;
        return e;
      };
      CKP(get(p > 0 ? w.D + (long long)pl.s[p] * bb : nullptr, bb));
      CKP(get(w.D + (long long)pl.e[p] * bb, bb));
      CKP(get(p > 0 ? w.BredIn + (long long)pl.q_s(p) * bb : nullptr, bb));
      if (ntip > 0) {
        vec_add_kernel<<<(ntip + 127) / 128, 128, 0, st>>>(ntip, src, red[m].Tt);
        BTA_COUNT(c);
      }
      src += (size_t)a * (a + 1);
      if (m == 0) {
        CKP(get(p > 0 ? w.RinRed + (long long)pl.q_s(p) * rs : nullptr, rs));
        CKP(get(w.RinRed + (long long)pl.q_e(p) * rs, rs));
      }
    }
  }
  return BTA_OK;
}

int PartRun::phase2() {
  const ModelDims& md = c->md;
  const int P = pl.P, nred = pl.nred;
  // ---- Phase 2: the reduced system (2P-1 boundary blocks), forward + tip + log-determinant
  for (int m = 0; m < 2; ++m) {
    cudaStream_t st = S[m][0];
    for (int q = 0; q < nred; ++q) CKP(chain_forward_step(red[m], q, st));
    CKP(chain_forward_end(red[m], st));
    CKP(chain_to_big(red[m], st));
    CKP(launch_logdet_partial(c, m == 0 ? CH_COND : CH_PRIOR, W[m].dvec, st));
  }
  // ---- Phase 2': reduced backward (x, Sigma of the boundary blocks, their traces)
  for (int m = 0; m < 2; ++m) {
    if (value_only && m == 1) break;
    cudaStream_t st = S[m][0];
    for (int q = nred - 1; q >= 0; --q) CKP(chain_backward_step(red[m], q, st));
    CKP(chain_to_big(red[m], st));
    for (int p = 1; p < P; ++p)
      if (local(p)) CKP(link(st, S[m][p]));
  }
  // ---- Phase 1': interior backward sweeps of the local partitions, concurrently
  int maxlen = 0;
  for (int p = 0; p < P; ++p)
    if (local(p)) maxlen = std::max(maxlen, pl.nint(p));
  for (int s = maxlen - 1; s >= 0; --s)
    for (int m = 0; m < 2; ++m) {
      if (value_only && m == 1) continue;
      for (int p = 0; p < P; ++p)
        if (local(p) && s < pc[m][p].nt) CKP(chain_backward_step(pc[m][p], s, S[m][p]));
    }
  // ---- join everything back onto s0; Phase B and the residual over the local time range
  for (int m = 0; m < 2; ++m)
    for (int p = 0; p < P; ++p) {
      if (local(p)) CKP(chain_to_big(pc[m][p], S[m][p]));
      CKP(link(S[m][p], s0));
    }
  CKP(cudaMemcpyAsync(W[0].x + (long long)md.nt * b, red[0].xT, a * sizeof(double), cudaMemcpyDeviceToDevice, s0));
  const int t_lo = nranks == 1 ? 0 : pl.s[rank], t_hi = nranks == 1 ? md.nt - 1 : pl.e[rank];
  CKP(launch_quad_stencil(c, W[0].x, t_lo, t_hi, s0));
  CKP(launch_residual(c, W[0].x, t_lo, t_hi, s0));
  return BTA_OK;
}

int PartRun::finish(bool timed) {
  const ModelDims& md = c->md;
  CKP(launch_scalars(c, s0));
  const int nout = 1 + md.d + 2 + 3 * md.d + md.k + 1;
  CKP(cudaMemcpyAsync(c->host_pinned + 64, c->small + L.out, nout * sizeof(double), cudaMemcpyDeviceToHost, s0));
  CKP(cudaMemcpyAsync(c->x_keep, W[0].x, md.N * sizeof(double), cudaMemcpyDeviceToDevice, s0));
  if (timed) CKP(cudaEventRecord(c->ev[8], s0));
  c->have_x = true;
  return BTA_OK;
}

}  // namespace

size_t part_ws_bytes(const bta_ctx* c) {
  const Plan pl = make_plan(c->md.nt, c->opt.partitions);
  Bump bp(nullptr);
  carve_part(bp, c->md, pl, true);
  carve_part(bp, c->md, pl, false);
  bp.take(c->md.N);
  return bp.off + 256;
}

int enqueue_gradient_partitioned(bta_ctx* c, void* ws, cudaStream_t s0, bool timed, bool value_only) {
  static thread_local PartRun run;   // ~20 Chain objects: keep them off the stack
  if (int rc = run.init(c, ws, s0, value_only, 0, 1); rc != BTA_OK) return rc;
  if (timed) CKP(cudaEventRecord(c->ev[0], s0));
  if (int rc = run.phase1(); rc != BTA_OK) return rc;
  if (int rc = run.phase2(); rc != BTA_OK) return rc;
  return run.finish(timed);
}

// ---- the multi-rank form (include/bta.h: inla_part_*)
extern "C" size_t bta_part_slab_doubles(const bta_ctx* c) {
  if (!c) return 0;
  const size_t bb = (size_t)c->md.b * c->md.b, rs = (size_t)(c->md.a + 1) * c->md.b;
  return 2 * (3 * bb + (size_t)c->md.a * (c->md.a + 1)) + 2 * rs;
}

extern "C" int inla_part_phase1(bta_ctx* c, const double* theta, int rank, int nranks, double* slab, void* ws,
                                void* stream) {
  if (!c || !theta || !slab || !ws) return bad("inla_part_phase1: null ctx, theta, slab or workspace");
  if (nranks < 2 || nranks > BTA_PMAX || rank < 0 || rank >= nranks) return bad("inla_part_phase1: need 2 <= nranks <= 8, 0 <= rank < nranks");
  if (c->store_mode != BTA_STORE_FACTOR || c->opt.partitions != nranks)
    return bad("inla_part_phase1: set BTA_STORE_FACTOR and bta_set_option(ctx, BTA_OPT_PARTITIONS, nranks) first (they size the workspace)");
  DeviceGuard guard(c->device);
  cudaStream_t s0 = (cudaStream_t)stream;
  memcpy(c->host_pinned, theta, c->md.d * sizeof(double));
  static thread_local PartRun run;
  if (int rc = run.init(c, ws, s0, false, rank, nranks); rc != BTA_OK) return rc;
  if (int rc = run.phase1(); rc != BTA_OK) return rc;
  if (int rc = run.pack(slab); rc != BTA_OK) return rc;
  CKP(cudaStreamSynchronize(s0));   // the slab is complete; host_pinned may be reused
  return BTA_OK;
}

extern "C" size_t bta_part_partial_doubles(const bta_ctx* c) { return c ? small_layout(c->md).Tt[0] : 0; }

extern "C" int inla_part_phase2(bta_ctx* c, int rank, int nranks, const double* gathered, double* partials, void* ws,
                                void* stream) {
  if (!c || !gathered || !partials || !ws) return bad("inla_part_phase2: null ctx, gathered slabs, partials or workspace");
  if (nranks < 2 || nranks > BTA_PMAX || rank < 0 || rank >= nranks || c->opt.partitions != nranks)
    return bad("inla_part_phase2: rank / nranks do not match phase 1");
  DeviceGuard guard(c->device);
  cudaStream_t s0 = (cudaStream_t)stream;
  static thread_local PartRun run;
  if (int rc = run.init(c, ws, s0, false, rank, nranks); rc != BTA_OK) return rc;
  if (int rc = run.unpack(gathered); rc != BTA_OK) return rc;
  if (int rc = run.phase2(); rc != BTA_OK) return rc;
  CKP(cudaMemcpyAsync(partials, c->small, run.L.Tt[0] * sizeof(double), cudaMemcpyDeviceToDevice, s0));
  CKP(cudaStreamSynchronize(s0));
  return BTA_OK;
}

extern "C" int inla_part_finish(bta_ctx* c, const double* partials, double* f, double* grad, void* stream) {
  if (!c || !partials) return bad("inla_part_finish: null ctx or partials");
  DeviceGuard guard(c->device);
  cudaStream_t s0 = (cudaStream_t)stream;
  const ModelDims& md = c->md;
  SmallLayout L = small_layout(md);
  CKP(cudaMemcpyAsync(c->small, partials, L.Tt[0] * sizeof(double), cudaMemcpyDeviceToDevice, s0));
  CKP(launch_scalars(c, s0));
  const int nout = 1 + md.d + 2 + 3 * md.d + md.k + 1;
  CKP(cudaMemcpyAsync(c->host_pinned + 64, c->small + L.out, nout * sizeof(double), cudaMemcpyDeviceToHost, s0));
  unsigned long long flag = 0;
  CKP(cudaMemcpyAsync(&flag, c->pivot_flag, sizeof flag, cudaMemcpyDeviceToHost, s0));
  CKP(cudaStreamSynchronize(s0));
  const double* o = c->host_pinned + 64;
  if (f) *f = o[0];
  if (grad) memcpy(grad, o + 1, md.d * sizeof(double));
  c->last_ld[0] = o[1 + md.d];
  c->last_ld[1] = o[1 + md.d + 1];
  c->last_parts.assign(o + 1 + md.d + 2, o + 1 + md.d + 2 + 3 * md.d);
  c->last_rss.assign(o + 1 + md.d + 2 + 3 * md.d, o + 1 + md.d + 2 + 3 * md.d + md.k);
  c->last_quad = o[1 + md.d + 2 + 3 * md.d + md.k];
  if (flag != ~0ull) {
    c->last_pivot = (long long)flag;
    bta_set_error("matrix is not positive definite on this rank (bta_last_pivot)");
    return BTA_ERR_NOTSPD;
  }
  c->last_pivot = 0;
  return BTA_OK;
}
