// One BTA chain (Q_p or Q_c) as the sweeps see it: pointers into caller-owned device memory.
#pragma once
#include "common.cuh"

// Middle partition of the time-domain partitioning (§III-C a): the interior
// blocks t = s+1 .. e-1 of a partition [s, e] are eliminated downwards BEFORE its two boundary blocks, so every interior
// block carries a fill coupling F~_t = Q~[s, t] to the top boundary s next to its coupling B_t to block t+1:
//   forward :  L_Ft = F~_t X_t^T,   D~_s -= L_Ft L_Ft^T,   [C~_s; r~_s] -= [L_Ct; z_t] L_Ft^T,   F~_{t+1} = -L_Ft L_Bt^T
//              (after the last interior block: Q~[e, s] = -L_Bt L_Ft^T goes to the reduced system)
//   backward:  H = L_Ft X_t,   Z_Bt -= Z_F{t+1}^T H,   Z_Ft = Sigma[s,t] = -(Z_F{t+1} G + Sigma[s,s] H + Sigma[T,s]^T E),
//              Z_Ct -= Sigma[T,s] H,   Z_Dt -= Z_Ft^T H,   x_t -= X_t^T L_Ft^T x_s.
struct Fill {
  double* LF = nullptr; long long lf_stride = 0;   // L_F(t), later Z_F(t), per interior block (local index)
  double* Ftil = nullptr;                          // scratch: F~_t of the current step (starts as B_s^T)
  double* H = nullptr;                             // scratch: H = L_F X (backward)
  double* Ds = nullptr;                            // forward: the top boundary block D~_s (reduced system)
  double* Rs = nullptr; int ld_rs = 0;             // forward: its stack rows [C~_s; r~_s]
  double* Bse = nullptr;                           // forward: where Q~[e, s] goes (reduced sub-diagonal block)
  const double* ZDs = nullptr;                     // backward: Sigma[s,s] (both triangles)
  const double* ZCs = nullptr;                     // backward: Sigma[T,s]  (a x b)
  const double* xs = nullptr; long long ld_xs = 0; // backward: x_s rows
  const double* ZFe = nullptr;                     // backward: Sigma[e,s] (stored [e][s]) for the last interior block
  int tb_first = -1;                               // global index of the pattern block B_s (trace of Z_F at t = s+1)
};

struct Chain {
  bta_ctx* c = nullptr;
  int chain = CH_COND;         // slot of the partial-sum buffers (CH_PRIOR / CH_COND)
  int b = 0, nt = 0, a = 0;
  int nr = 0;                  // right-hand-side rows carried through the sweeps
  bool factor_blocks = true;   // forward: POTRF/TRTRI of the diagonal blocks, L_B, Schur updates
  bool arrow_rows = false;     // forward: the stack holds the a arrow rows C_t, factored to L_Ct
  bool arrow_given = false;    // the arrow factor rows L_Ct already exist (solve with a stored factor)
  bool tip_chol = true;        // forward: factor the reduced tip (else L_T is given)
  bool zero_upper = false;     // forward: clear the strict upper triangle of D_t first
  bool selinv = false;         // backward: selected inversion
  bool contract = false;       // backward: accumulate the Eq. 7 traces per block (fused gradient)
  bool selinv_inplace = false; // backward: copy Z_D / Z_C back over D / C (bta_selinv)
  bool carry = false;          // carry mode (a7): D(t) keeps D_t - S_{t-1}; X_t, L_Bt live in Xs / LBs and are rebuilt
  int which = BTA_COND;        // carry mode: which matrix B_t is re-assembled for
  // Sub-chain of a two-way (twisted) elimination: local block s is global time block t0 + tdir * s; with
  // tail_coupling the last local block also couples (through B(nt-1)) to a separator block eliminated later.
  int t0 = 0, tdir = 1;
  bool tail_coupling = false;
  bool transposeB = false;     // the coupling blocks of this chain are B^T (down chain); carry mode re-assembly
  bool tt_zero = false;        // forward_begin: start the tip accumulator from zero (the up chain carries T)
  const double* sep_x = nullptr;   // backward: x, Z_D, Z_C of the separator (the "next" block of local block nt-1)
  const double* sep_ZD = nullptr;
  const double* sep_ZC = nullptr;
  cudaStream_t hi = nullptr;   // optional high-priority companion stream for the small kernels of this chain
  bool on_small = false;       // which lane the chain's work currently ends on
  bool lanes_bwd = true;       // use the small lane in the backward sweep too
  int trace_id = -1;           // BTA_TRACE label of this chain
  cudaStream_t xs = nullptr;   // optional side stream: work of a forward step that is off its dependent chain
  // Forward pipelining (sweep.cu: chain_forward_step): three events of this chain -- [0] the top-left part of the next
  // diagonal block has its Schur update, [1] L_B of this step is complete, [2] all products of this step are done.
  cudaEvent_t* pipe_ev = nullptr;
  bool pipe_armed = false;     // the previous step recorded pipe_ev (its products were issued in split form)
  // Rows stream: the arrow / right-hand-side rows of a forward step (R~_t, R^_t = [L_Ct; z_t], tip updates) and the trace
  // contractions of a backward step do not feed the next block's factorisation or selected inversion, so (factor mode)
  // they run on this third stream, one step behind the chain, instead of sitting in its dependent launch sequence.
  // pipe_ev[3], [4]: the contractions of an even / odd backward step have read their Z buffers.
  cudaStream_t rs = nullptr;
  bool rows_pending = false;   // work is outstanding on rs (chain_to_big joins it)
  // Solve stream: the upper solve of a backward step (Eqs. 3-5: u = z_t - L_Bt^T x_{t+1} - L_Ct^T x_T, x_t = X_t^T u) reads
  // only forward results and x_{t+1}, never the selected inverse, so (factor mode) its three to five small kernels run
  // on this stream, ahead of the chain, with their own partial-sum scratch `part2`; the chain only waits, before Z_Bt
  // overwrites the slot of L_Bt, for the solve step that read it.
  // The arrow products E = L_Ct X_t and Z_T E of the selected inversion read only forward results as well: they run on
  // the same stream into a ring of two buffers (step parity), one step ahead of the chain; pipe_ev[5 + parity] says
  // "ready", pipe_ev[7 + parity] "consumed".
  cudaStream_t ss = nullptr;
  bool solve_pending = false;  // work is outstanding on ss (chain_to_big joins it)
  double* part2 = nullptr;
  double *Ebuf2[2] = {nullptr, nullptr}, *Ybuf2[2] = {nullptr, nullptr};
  bool ey_used[2] = {false, false};
  // So do G = L_Bt X_t (into a ring of two b x b buffers) and X_t^T X_t (straight into the step's Z_D buffer, once the
  // next step's Z_B product and the traces two steps back have read it): the dependent chain of a backward step is then
  // Z_C, Z_B = -Z_D{t+1} G - ..., Z_D -= Z_B^T G.  pipe_ev[9 + parity] ready, [11 + parity] G consumed, [13 + parity]
  // Z_D buffer of that parity read.
  double* Gm2[2] = {nullptr, nullptr};
  bool g_used[2] = {false, false}, zd_read[2] = {false, false};
  cudaStream_t gs = nullptr;   // the stream G and X^T X run on (the solve stream carries ten kernels per step already)
  bool g_pending = false;      // work is outstanding on gs (chain_to_big joins it)
  bool tr_armed[2] = {false, false};
  // Host-staged carries (BTA_STORE_HOST): the diagonal-block slots are a ring of `ring` device blocks
  // (local block s lives in slot s % ring); each carry D_s - S_{s-1} is copied to pinned host memory (hostD + s b^2) on
  // the copy stream `cs` during the forward sweep and streamed back `ring` steps ahead in the backward sweep.
  // ring_ev[slot]: the last copy from / into that slot has finished.
  int ring = 0;
  double* hostD = nullptr;
  cudaStream_t cs = nullptr;
  cudaEvent_t* ring_ev = nullptr;
  double* Dp(int s) const {
    return dmap ? dmap[s] : (ring ? D + (long long)(s % ring) * b * b : D + s * d_stride);
  }
  // Reduced system of the partitioning: the local blocks are the boundary blocks of the partitions -- their global time
  // index, the global index of the pattern block between local s and s+1 (-1: a fill block, no trace), and their
  // device pointers come from host tables.
  const int* tmap = nullptr;
  const int* bmap = nullptr;
  double* const* dmap = nullptr;
  Fill* fill = nullptr;        // this chain is the interior of a middle partition
  int tg(int s) const { return tmap ? tmap[s] : t0 + tdir * s; }
  int tB(int s) const { return bmap ? bmap[s] : (tdir > 0 ? tg(s) : tg(s) - 1); }   // sub-diagonal block between s, s+1

  int P() const { return (arrow_rows ? a : 0) + nr; }
  bool arrow() const { return arrow_rows || arrow_given; }

  double* D = nullptr;    long long d_stride = 0;      // D(t) = D + t * d_stride   (b x b, ld b)
  double* Bin = nullptr;  double* Bout = nullptr; long long b_stride = 0;
  // forward stack: rows [arrow rows | rhs rows] of time block t
  double* Rin = nullptr;  long long rin_stride = 0;  int ld_rin = 0;
  double* Rout = nullptr; long long rout_stride = 0; int ld_rout = 0;   // [L_Ct | z_t]
  double* Rtmp = nullptr;                                               // P x b scratch, or NULL: in place in Rin
  const double* LCgiven = nullptr; long long lc_stride = 0;             // arrow_given: L_Ct = LCgiven + t * lc_stride
  double* T = nullptr; int ldT = 0;                                     // tip (a x a)
  const double* rhs_tip = nullptr; int rhs_tip_stride = 0;              // rhs_tip[r * stride + p]
  // scratch
  double *W1 = nullptr, *W2 = nullptr, *W3 = nullptr;                   // b x b each
  double *Xs = nullptr, *LBs = nullptr, *Bs = nullptr;                  // carry mode: X_t, L_Bt, assembled B_t
  double* part = nullptr;                                               // skinny_nn partial sums
  double *ubuf = nullptr, *Ebuf = nullptr, *Ybuf = nullptr;             // [nr][b], [a][b], [a][b]
  double* ZC[2] = {nullptr, nullptr};                                   // [a][b] ping-pong
  double* dvec = nullptr;                                               // diag(L), N doubles, or NULL
  double *Tt = nullptr, *LT = nullptr, *zT = nullptr, *xT = nullptr, *ZT = nullptr;
  // backward outputs
  double* xout = nullptr; long long ld_x = 0;                           // x rows: xout + r * ld_x + t * b
  double* Cout = nullptr; long long cout_stride = 0;                    // selinv_inplace: Z_Ct destination
};

// phase 0: the whole POTRF + TRTRI; 1: only the first half of the top level (A11); 2: everything but that half
cudaError_t potrf_inv(bta_ctx* c, Chain* lanes, double* A, int ld, int lo, int hi, double* T1, double* T2,
                      double* diagL, long long grow0, cudaStream_t st, int phase = 0);
int potrf_split(int n);  // size of the first half of the top level of potrf_inv on an n x n block
cudaError_t chain_to_big(Chain& ch, cudaStream_t big);  // join the small lane back into the chain's main stream
cudaError_t chain_forward(Chain& ch, cudaStream_t st);
cudaError_t chain_forward_begin(Chain& ch, cudaStream_t st);
cudaError_t chain_forward_step(Chain& ch, int t, cudaStream_t st);
cudaError_t chain_forward_end(Chain& ch, cudaStream_t st);
cudaError_t chain_backward_step(Chain& ch, int t, cudaStream_t st);
cudaError_t separator_merge_forward(Chain& up, Chain& dn, Chain& cs, cudaStream_t st);
cudaError_t chain_backward(Chain& ch, cudaStream_t st);
