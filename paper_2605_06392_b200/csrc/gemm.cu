// FP64 tensor-core GEMM for sm_100a: C = alpha * op(A) op(B) + beta * C (row-major).
//
// The dense b x b block products of the BTA sweeps (Algorithm 1's TRSM/SYRK steps, and
// the selected-inversion products) all run through this kernel.  sm_100a has no
// tcgen05 f64 kind; the FP64 tensor path is warp-level `mma.sync.m8n8k4.f64` (SASS DMMA.8x8x4).
// Operands are staged in shared memory by a 3-stage (template parameter) cp.async (LDGSTS) pipeline in layouts chosen so the
// 64-bit fragment loads are bank-conflict-free (leading dimension = 4 mod 16 doubles); accumulators live
// in registers.  Triangular operands are exploited by restricting the k-range per output tile
// (KLO_*/KHI_*), symmetric outputs by computing the lower tiles only (OUT_LOWER*).
#include <algorithm>

#include "common.cuh"

namespace {

constexpr int KPAD = 4;  // leading dimensions are == 4 (mod 16) doubles

// Diagnostic CTA timeline (bta_debug_cta_trace; null in production): one record per CTA that did work,
// {start ns, end ns, smid | BM << 16 | mode << 28, k-range | M << 32} from %globaltimer.
__device__ unsigned long long* g_cta_trace = nullptr;
__device__ unsigned int g_cta_cap = 0;
__device__ unsigned int g_cta_n = 0;
__device__ __forceinline__ unsigned long long global_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, int src_bytes) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async8(void* smem, const void* gmem, int src_bytes) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(s), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}

// Split barrier (mbarrier in shared memory): arrive early, wait late, so the barrier latency hides behind DMMAs.
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
  unsigned a = (unsigned)__cvta_generic_to_shared(bar);
  asm volatile("mbarrier.init.shared.b64 [%0], %1;\n" ::"r"(a), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {
  unsigned a = (unsigned)__cvta_generic_to_shared(bar);
  asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.shared.b64 st, [%0];\n}\n" ::"r"(a) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  unsigned a = (unsigned)__cvta_generic_to_shared(bar);
  asm volatile(
      "{\n.reg .pred p;\nWAIT_LOOP:\nmbarrier.try_wait.parity.shared.b64 p, [%0], %1;\n@!p bra WAIT_LOOP;\n}\n" ::"r"(a),
      "r"(parity)
      : "memory");
}

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

// One operand tile (ROWS rows of the output dimension x BK of k) -> shared memory.
//  KM = false: global is [row][k] (k contiguous); smem [ROWS][BK+KPAD]
//  KM = true : global is [k][row] (row contiguous); smem [BK][ROWS+KPAD]
template <int ROWS, bool KM, int NT, int BK>
__device__ __forceinline__ void load_tile(double* sm, const double* __restrict__ g, int ld, int row0, int nrows,
                                          int k0, int kend, bool vec, int tid) {
  constexpr int CHUNKS = ROWS * BK / 2;
#pragma unroll
  for (int c = tid; c < CHUNKS; c += NT) {
    int r, k;
    double* dst;
    const double* src;
    int n_ok;  // valid elements of this 2-element chunk (0, 1, 2)
    if (!KM) {
      r = c / (BK / 2);
      k = (c % (BK / 2)) * 2;
      dst = sm + r * (BK + KPAD) + k;
      int gr = row0 + r, gk = k0 + k;
      n_ok = (gr < nrows) ? max(0, min(2, kend - gk)) : 0;
      src = g + (long long)gr * ld + gk;
    } else {
      k = c / (ROWS / 2);
      r = (c % (ROWS / 2)) * 2;
      dst = sm + k * (ROWS + KPAD) + r;
      int gr = row0 + r, gk = k0 + k;
      n_ok = (gk < kend) ? max(0, min(2, nrows - gr)) : 0;
      src = g + (long long)gk * ld + gr;
    }
    if (vec) {
      cp_async16(dst, n_ok ? src : g, n_ok * 8);
    } else {
      cp_async8(dst, n_ok > 0 ? src : g, n_ok > 0 ? 8 : 0);
      cp_async8(dst + 1, n_ok > 1 ? src + 1 : g, n_ok > 1 ? 8 : 0);
    }
  }
}

// Fast path of load_tile for a tile that lies fully inside the matrix with a full BK of k and 16-byte
// alignment: one running global pointer per operand, constant strides, no predicates.
//  KM = false: thread's chunk i sits at row (tid / (BK/2)) + i * (NT / (BK/2)), k = (tid % (BK/2)) * 2
//  KM = true : chunk i sits at k = tid / (ROWS/2) + i * (NT / (ROWS/2)), row = (tid % (ROWS/2)) * 2
template <int ROWS, bool KM, int NT, int BK>
__device__ __forceinline__ void load_tile_fast(double* sm_thread, const double* __restrict__ g_thread, long long ld) {
  constexpr int CHUNKS = ROWS * BK / 2;
  static_assert(CHUNKS % NT == 0, "tile chunks must divide evenly over the CTA");
  constexpr int PER = CHUNKS / NT;
  if (!KM) {
    static_assert(NT % (BK / 2) == 0, "row stride");
    constexpr int RSTEP = NT / (BK / 2);
#pragma unroll
    for (int i = 0; i < PER; ++i)
      cp_async16(sm_thread + i * RSTEP * (BK + KPAD), g_thread + (long long)i * RSTEP * ld, 16);
  } else {
    static_assert(NT % (ROWS / 2) == 0 || (ROWS / 2) % NT == 0, "k stride");
    if (NT >= ROWS / 2) {
      constexpr int KSTEP = NT / (ROWS / 2) > 0 ? NT / (ROWS / 2) : 1;
#pragma unroll
      for (int i = 0; i < PER; ++i)
        cp_async16(sm_thread + i * KSTEP * (ROWS + KPAD), g_thread + (long long)i * KSTEP * ld, 16);
    } else {
      constexpr int SPLIT = (ROWS / 2) / NT > 0 ? (ROWS / 2) / NT : 1;  // chunks of one k-row handled per thread
#pragma unroll
      for (int i = 0; i < PER; ++i)
        cp_async16(sm_thread + (i / SPLIT) * (ROWS + KPAD) + (i % SPLIT) * NT * 2,
                   g_thread + (long long)(i / SPLIT) * ld + (i % SPLIT) * NT * 2, 16);
    }
  }
}

template <int BM, int BN, int WM, int WN, bool A_KM, bool B_KM, int BK, int STAGES>
struct Cfg {
  static constexpr int NWM = BM / WM, NWN = BN / WN;
  static constexpr int NT = NWM * NWN * 32;
  static constexpr int A_ST = A_KM ? BK * (BM + KPAD) : BM * (BK + KPAD);
  static constexpr int B_ST = B_KM ? BK * (BN + KPAD) : BN * (BK + KPAD);
  static constexpr int SMEM = (2 + STAGES * (A_ST + B_ST)) * (int)sizeof(double);
};

// CLIP: per-warp clipping of the k-range (see below); measured to pay in the 64x64-tile class only (+2 % on triangular
// products at b = 2304; the 128x128 and 32x32 classes lose 1-2 % to the extra branch), so only that class carries it.
template <int BM, int BN, int WM, int WN, bool A_KM, bool B_KM, int MINB, int BK, int STAGES, bool TRACE = false,
          bool CLIP = (BM == 64)>
__global__ void __launch_bounds__(Cfg<BM, BN, WM, WN, A_KM, B_KM, BK, STAGES>::NT, MINB) gemm_kernel(GemmArgs g) {
  using C_ = Cfg<BM, BN, WM, WN, A_KM, B_KM, BK, STAGES>;
  constexpr int NT = C_::NT;
  extern __shared__ __align__(16) double smem[];
  if constexpr (BM == 32) {  // latency-bound class: launched programmatically (launch_cfg)
    pdl_wait();
    pdl_launch_dependents();
  }
  unsigned long long* bar = reinterpret_cast<unsigned long long*>(smem);  // 16 bytes reserved
  double* As = smem + 2;
  double* Bs = As + STAGES * C_::A_ST;

  const double* __restrict__ A = g.A;
  const double* __restrict__ B = g.B;
  double* __restrict__ C = g.C;
  int M = g.M, N = g.N, K = g.K;
  if (g.subs) {
    GemmSub s = g.subs[blockIdx.z];
    A += s.offA;
    B += s.offB;
    C += s.offC;
    M = s.M;
    N = s.N;
    K = s.K;
  }
  // Tile order: CTAs are dispatched x-fastest.  With a restricted k-range the work per tile varies by up to 32x;
  // the tiles are enumerated heaviest-first (the heavy tile column / row is the slow grid dimension), so the last,
  // partially filled wave consists of the lightest tiles.
  // Within that order the slow index is regrouped: `group` consecutive slow tile rows are swept together (slow index
  // fastest inside a group), so the ~148 co-resident CTAs form a (group x 148/group) patch of the tile grid that
  // shares `group` panels of one operand and 148/group of the other, instead of 4.6 x 32: fewer DRAM re-reads.
  int slow = blockIdx.y, fastx = blockIdx.x;
  if (g.group > 1) {
    const int per = g.group * (int)gridDim.x;
    const int lin = slow * (int)gridDim.x + fastx;
    const int grp = lin / per, within = lin - grp * per;
    const int gsz = min(g.group, (int)gridDim.y - grp * g.group);
    slow = grp * g.group + within % gsz;
    fastx = within / gsz;
  }
  int tm = slow, tn = fastx;
  if (g.klo == KLO_N0) {
    tm = fastx;
    tn = slow;
  } else if (g.khi == KHI_NEND) {
    tm = fastx;
    tn = (int)gridDim.y - 1 - slow;
  } else if (g.khi == KHI_MEND) {
    tm = (int)gridDim.y - 1 - slow;
  }
  const int m0 = tm * BM, n0 = tn * BN;
  if (m0 >= M || n0 >= N) return;
  if (g.out != OUT_FULL && n0 > m0 + BM - 1) return;  // tile entirely above the diagonal

  int kbeg = 0, kend = K;
  if (g.klo == KLO_N0) kbeg = n0;
  if (g.klo == KLO_M0) kbeg = m0;
  if (g.khi == KHI_NEND) kend = min(K, n0 + BN);
  if (g.khi == KHI_MEND) kend = min(K, m0 + BM);
  kbeg = (kbeg / BK) * BK;
  // TRACE instantiations only (bta_debug_cta_trace): measured, a run-time test here costs the production kernel 1.5 %
  unsigned long long t_begin = 0ull;
  if constexpr (TRACE) t_begin = threadIdx.x == 0 ? global_ns() : 0ull;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm0 = (warp / C_::NWN) * WM, wn0 = (warp % C_::NWN) * WN;
  const int gid = lane >> 2, tig = lane & 3;

  const bool vecA = ((g.lda & 1) == 0) && ((((uintptr_t)A) & 15) == 0);
  const bool vecB = ((g.ldb & 1) == 0) && ((((uintptr_t)B) & 15) == 0);

  double acc[WM / 8][WN / 8][2];
#pragma unroll
  for (int i = 0; i < WM / 8; ++i)
#pragma unroll
    for (int j = 0; j < WN / 8; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  const int nk = (kend > kbeg) ? (kend - kbeg + BK - 1) / BK : 0;
  // Per-warp clipping of the k-range: the CTA's range [kbeg, kend) is tile-granular; inside a tile that touches the
  // diagonal of a triangular operand (or of a lower-only output) a warp's WM x WN sub-tile needs less -- e.g. with
  // KHI_NEND the columns [n, n + WN) need only k < n + WN.  A warp outside its live k-tiles issues no fragment loads
  // and no DMMAs (the tensor pipe is the bottleneck: the other warps of the SM sub-partition take the issue slots),
  // but keeps taking part in the stage barriers.  Saves ~2 % of the DMMAs of a triangular b^3 product.
  int kw_lo = kbeg, kw_hi = kend;
  if (g.klo == KLO_N0) kw_lo = max(kw_lo, n0 + wn0);
  if (g.klo == KLO_M0) kw_lo = max(kw_lo, m0 + wm0);
  if (g.khi == KHI_NEND) kw_hi = min(kw_hi, n0 + wn0 + WN);
  if (g.khi == KHI_MEND) kw_hi = min(kw_hi, m0 + wm0 + WM);
  if (g.out != OUT_FULL && n0 + wn0 > m0 + wm0 + WM - 1) kw_hi = kw_lo;  // sub-tile entirely above the diagonal
  const int itw_lo = CLIP ? (kw_lo - kbeg) / BK : 0;
  const int itw_hi = CLIP ? (kw_hi > kw_lo ? (kw_hi - kbeg + BK - 1) / BK : itw_lo) : nk;

  // per-thread origins of the fast path (interior tile, aligned operands)
  const bool fast = vecA && vecB && (m0 + BM <= M) && (n0 + BN <= N);
  const double* gA;
  const double* gB;
  int sA, sB;  // offsets (doubles) of this thread's first chunk inside a stage
  if (!A_KM) {
    const int r = tid / (BK / 2), k = (tid % (BK / 2)) * 2;
    gA = A + (long long)(m0 + r) * g.lda + kbeg + k;
    sA = r * (BK + KPAD) + k;
  } else {
    const int k = tid / (BM / 2), r = (tid % (BM / 2)) * 2;
    gA = A + (long long)(kbeg + k) * g.lda + m0 + r;
    sA = k * (BM + KPAD) + r;
  }
  if (!B_KM) {
    const int r = tid / (BK / 2), k = (tid % (BK / 2)) * 2;
    gB = B + (long long)(n0 + r) * g.ldb + kbeg + k;
    sB = r * (BK + KPAD) + k;
  } else {
    const int k = tid / (BN / 2), r = (tid % (BN / 2)) * 2;
    gB = B + (long long)(kbeg + k) * g.ldb + n0 + r;
    sB = k * (BN + KPAD) + r;
  }
  const long long stepA = A_KM ? (long long)BK * g.lda : BK, stepB = B_KM ? (long long)BK * g.ldb : BK;

  auto issue = [&](int it) {
    if (it < nk) {
      const int s = it % STAGES;
      const int k0 = kbeg + it * BK;
      if (fast && k0 + BK <= kend) {
        load_tile_fast<BM, A_KM, NT, BK>(As + s * C_::A_ST + sA, gA + it * stepA, g.lda);
        load_tile_fast<BN, B_KM, NT, BK>(Bs + s * C_::B_ST + sB, gB + it * stepB, g.ldb);
      } else {
        load_tile<BM, A_KM, NT, BK>(As + s * C_::A_ST, A, g.lda, m0, M, k0, kend, vecA, tid);
        load_tile<BN, B_KM, NT, BK>(Bs + s * C_::B_ST, B, g.ldb, n0, N, k0, kend, vecB, tid);
      }
    }
    cp_async_commit();
  };

#pragma unroll
  for (int s = 0; s < STAGES - 1; ++s) issue(s);
  if (tid == 0) mbar_init(bar, NT);
  cp_async_wait<STAGES - 2>();
  __syncthreads();  // stage 0 is visible, the mbarrier is initialised

  // Per k-tile: [k-step 0: DMMAs, then the refill of the stage consumed one iteration ago] ... [last k-step: this
  // thread's last reads of the stage, wait for its own copies of the next stage, ARRIVE, DMMAs, then WAIT].  When all
  // NT threads have arrived, the next stage is visible and the current one is free -- one split barrier per k-tile
  // whose latency is covered by the last k-step's DMMAs.  (The refill is issued after the first k-step, not right
  // after the barrier: address arithmetic there would idle the tensor pipe of every scheduler at once.)
  for (int it = 0; it < nk; ++it) {
    const double* as = As + (it % STAGES) * C_::A_ST;
    const double* bs = Bs + (it % STAGES) * C_::B_ST;
    const bool live = !CLIP || (it >= itw_lo && it < itw_hi);  // warp-uniform
#pragma unroll
    for (int kk = 0; kk < BK; kk += 4) {
      double af[WM / 8], bf[WN / 8];
      if (live) {
#pragma unroll
        for (int i = 0; i < WM / 8; ++i) {
          int m = wm0 + i * 8 + gid, k = kk + tig;
          af[i] = A_KM ? as[k * (BM + KPAD) + m] : as[m * (BK + KPAD) + k];
        }
#pragma unroll
        for (int j = 0; j < WN / 8; ++j) {
          int n = wn0 + j * 8 + gid, k = kk + tig;
          bf[j] = B_KM ? bs[k * (BN + KPAD) + n] : bs[n * (BK + KPAD) + k];
        }
      }
      if (kk == BK - 4) {
        cp_async_wait<STAGES - 2>();
        mbar_arrive(bar);
      }
      if (live) {
#pragma unroll
        for (int i = 0; i < WM / 8; ++i)
#pragma unroll
          for (int j = 0; j < WN / 8; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
      }
      if (kk == 0) issue(it + STAGES - 1);
      if (kk == BK - 4) mbar_wait(bar, (unsigned)(it & 1));
    }
  }
  cp_async_wait<0>();

  // epilogue: C = alpha * acc + beta * C (guarded; optional lower mask / mirrored write)
  const double alpha = g.alpha, beta = g.beta;
  const int ldc = g.ldc;
  const bool lower = g.out != OUT_FULL, mirror = g.out == OUT_LOWER_MIRROR;
#pragma unroll
  for (int i = 0; i < WM / 8; ++i) {
    const int row = m0 + wm0 + i * 8 + gid;
    if (row >= M) continue;
#pragma unroll
    for (int j = 0; j < WN / 8; ++j) {
      const int col = n0 + wn0 + j * 8 + tig * 2;
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int c = col + e;
        if (c >= N) continue;
        if (lower && c > row) continue;
        double* p = C + (long long)row * ldc + c;
        double v = alpha * acc[i][j][e];
        if (beta != 0.0) v += beta * (*p);
        *p = v;
        if (mirror && c < row) C[(long long)c * ldc + row] = v;
      }
    }
  }
  if constexpr (TRACE) {
    unsigned long long* const cta_trace = g_cta_trace;
    const unsigned idx = (cta_trace && tid == 0) ? atomicAdd(&g_cta_n, 1u) : 0xFFFFFFFFu;
    if (cta_trace && tid == 0 && idx < g_cta_cap) {
      unsigned smid;
      asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
      unsigned long long* r = cta_trace + 4ull * idx;
      r[0] = t_begin;
      r[1] = global_ns();
      r[2] = (unsigned long long)smid | ((unsigned long long)BM << 16) | ((unsigned long long)g.mode << 28);
      r[3] = (unsigned long long)(unsigned)(kend - kbeg) | ((unsigned long long)(unsigned)M << 32);
    }
  }
}

// Element-exact flop count of one launch: 2 * sum over the written (m, n) of the length of the k-range that element
// needs (triangular operands: KLO_* / KHI_*; lower-only outputs: m >= n).  Batched launches are not used by the sweeps.
double gemm_alg_flop(const GemmArgs& g) {
  double total = 0.0;
  for (int n = 0; n < g.N; ++n) {
    // rows m in [mlo, M) are written for this column
    const int mlo = g.out != OUT_FULL ? n : 0;
    if (mlo >= g.M) continue;
    const double rows = g.M - mlo;
    auto series = [](double first, double last, double cnt) { return cnt > 0 ? 0.5 * (first + last) * cnt : 0.0; };
    if (g.klo == KLO_M0 && g.khi != KHI_MEND) {          // len(m) = H - m for m < H
      const int H = g.khi == KHI_NEND ? std::min(g.K, n + 1) : g.K;
      const int mhi = std::min(g.M, H);
      if (mhi > mlo) total += series(H - mlo, H - (mhi - 1), mhi - mlo);
    } else if (g.khi == KHI_MEND && g.klo != KLO_M0) {   // len(m) = min(K, m + 1) - L for m + 1 > L
      const int L = g.klo == KLO_N0 ? n : 0;
      const int m0 = std::max(mlo, L);                   // first row with a non-empty range
      const int msat = std::max(m0, g.K - 1);            // from here on the range is [L, K)
      if (g.M > m0) {
        const int mramp = std::min(g.M, msat);
        if (mramp > m0) total += series(m0 + 1 - L, mramp - L, mramp - m0);
        if (g.M > msat && g.K > L) total += (double)(g.M - msat) * (g.K - L);
      }
    } else if (g.klo == KLO_M0 && g.khi == KHI_MEND) {   // one k per element
      total += std::max(0, std::min(g.M, g.K) - mlo);
    } else {
      const int hi = g.khi == KHI_NEND ? std::min(g.K, n + 1) : g.K;
      const int lo = g.klo == KLO_N0 ? n : 0;
      if (hi > lo) total += rows * (hi - lo);
    }
  }
  return 2.0 * total * (g.subs ? g.nsub : 1);
}

template <int BM, int BN, int WM, int WN, bool A_KM, bool B_KM, int MINB, int BK, int STAGES, bool TRACE>
cudaError_t launch_cfg(const GemmArgs& g, cudaStream_t st) {
  using C_ = Cfg<BM, BN, WM, WN, A_KM, B_KM, BK, STAGES>;
  auto kern = gemm_kernel<BM, BN, WM, WN, A_KM, B_KM, MINB, BK, STAGES, TRACE>;
  static unsigned long long attr_done = 0ull;  // per instantiation, one bit per device
  if (cudaError_t e = optin_smem(kern, C_::SMEM, &attr_done); e != cudaSuccess) return e;
  const int tilesM = (g.M + BM - 1) / BM, tilesN = (g.N + BN - 1) / BN;
  const bool swap = g.klo == KLO_N0 || g.khi == KHI_NEND;  // heavy-first enumeration (see the kernel)
  dim3 grid(swap ? tilesM : tilesN, swap ? tilesN : tilesM, g.subs ? g.nsub : 1);
  GemmArgs ga = g;
  if (ga.group > 1) {  // equal-sized groups of at most `group` slow tile rows (18 rows -> 9 + 9, not 16 + 2)
    const int ngroups = ((int)grid.y + ga.group - 1) / ga.group;
    ga.group = ((int)grid.y + ngroups - 1) / ngroups;
  }
  KTimeScope kt(BM == 128 ? BTA_KC_GEMM_BIG : (BM == 64 ? BTA_KC_GEMM_SMALL : BTA_KC_GEMM_TINY), st,
                g_ktime_on ? gemm_alg_flop(g) : 0.0, 0.0);
  if (BM == 32 && (g_pdl == 1 || g_pdl == 2)) return launch_pdl(kern, grid, dim3(C_::NT), (size_t)C_::SMEM, st, ga);
  kern<<<grid, C_::NT, C_::SMEM, st>>>(ga);
  return cudaGetLastError();
}

template <int BM, int BN, int WM, int WN, int MINB, int BK, int STAGES = 3, bool TRACE = false>
cudaError_t launch_mode(const GemmArgs& g, cudaStream_t st) {
  switch (g.mode) {
    case GEMM_NN: return launch_cfg<BM, BN, WM, WN, false, true, MINB, BK, STAGES, TRACE>(g, st);
    case GEMM_NT: return launch_cfg<BM, BN, WM, WN, false, false, MINB, BK, STAGES, TRACE>(g, st);
    case GEMM_TN: return launch_cfg<BM, BN, WM, WN, true, true, MINB, BK, STAGES, TRACE>(g, st);
  }
  return cudaErrorInvalidValue;
}

}  // namespace

// Tile-choice parameters (bta_set_option: BTA_OPT_TILE_THRESH / BTA_OPT_TILE_WAVES; process-global)
int g_pdl = 3;   // BTA_OPT_PDL: 0 off, 1 leaves and 32x32-tile GEMMs, 2 the GEMMs only, 3 the leaves only (measured best)
long long g_tile_thresh = 180;  // fewer big tiles than this: 64x64 tiles (measured)
int g_tile_waves = 1;           // 1: also prefer 64x64 tiles where the last wave of big tiles would be mostly empty

// Tile choice: 128x128 (16 warps, 32x32 per warp) once the problem fills the chip with big tiles,
// else 64x64 (4 warps, 32x32 per warp, three CTAs per SM), and 32x32 for the latency-bound launches.
namespace {
long long big_tiles(const GemmArgs& g) {
  long long tiles128 = (long long)((g.M + 127) / 128) * ((g.N + 127) / 128) * (g.subs ? g.nsub : 1);
  if (g.out != OUT_FULL) tiles128 = tiles128 / 2 + 1;
  return tiles128;
}
constexpr long long kTinyThreshold = 148;  // at most this many 64x64 tiles: 32x32 tiles
}  // namespace

// Small tiles (64x64, three CTAs per SM) for launches of fewer than ~1.2 waves of big tiles, and wherever the last,
// partially filled wave of big tiles would cost more than the small tiles' lower rate (0.97 of the big tile's):
// e.g. the lower-only products at b = 3072 are 300 big tiles = 2.03 waves (3 waves: 68 %) but 1176 small ones =
// 2.65 waves of 444.
bool gemm_uses_small_tiles(const GemmArgs& g) {
  const long long t128 = big_tiles(g);
  if (t128 < g_tile_thresh) return true;
  if (!g_tile_waves) return false;
  const long long nb = g.subs ? g.nsub : 1;
  const long long m64 = (g.M + 63) / 64, n64 = (g.N + 63) / 64;
  const long long t64 = (g.out != OUT_FULL ? std::min(m64, n64) * (std::min(m64, n64) + 1) / 2 : m64 * n64) * nb;
  const long long m128 = (g.M + 127) / 128, n128 = (g.N + 127) / 128;
  const long long x128 =
      (g.out != OUT_FULL ? std::min(m128, n128) * (std::min(m128, n128) + 1) / 2 : m128 * n128) * nb;
  const double e128 = (double)x128 / (double)(((x128 + 147) / 148) * 148);
  const double e64 = 0.97 * (double)t64 / (double)(((t64 + 443) / 444) * 444);
  return e64 > e128 + 0.03;
}

namespace {
// Latency-bound launches (the deep levels of the POTRF+TRTRI recursion: a few dozen 64x64 tiles, one dependent kernel
// after the other): 32x32 tiles (4 warps, 16x16 per warp) shorten each CTA's k-loop fourfold (4 DMMAs per k-step and
// warp instead of 16) and spread the product over four times as many CTAs.
bool gemm_uses_tiny_tiles(const GemmArgs& g) {
  long long t64 = (long long)((g.M + 63) / 64) * ((g.N + 63) / 64) * (g.subs ? g.nsub : 1);
  if (g.out != OUT_FULL) t64 = t64 / 2 + 1;
  return t64 <= kTinyThreshold;
}
}  // namespace

static bool g_trace_host = false;  // set while bta_debug_cta_trace is armed: launch the TRACE twins of the default tiles

cudaError_t launch_gemm(const GemmArgs& g0, cudaStream_t st) {
  if (g0.M <= 0 || g0.N <= 0) return cudaSuccess;
  GemmArgs g = g0;
  g.group = 16;  // tile-order grouping (sweep over 0/4/8/12/16/32)
  if (g_trace_host) {
    if (!gemm_uses_small_tiles(g)) return launch_mode<128, 128, 32, 32, 1, 16, 3, true>(g, st);
    if (gemm_uses_tiny_tiles(g)) return launch_mode<32, 32, 16, 16, 4, 16, 3, true>(g, st);
    return launch_mode<64, 64, 32, 32, 3, 16, 3, true>(g, st);
  }
  if (!gemm_uses_small_tiles(g)) return launch_mode<128, 128, 32, 32, 1, 16>(g, st);  // 16 warps, 32x32 per warp
  if (gemm_uses_tiny_tiles(g)) return launch_mode<32, 32, 16, 16, 4, 16>(g, st);
  return launch_mode<64, 64, 32, 32, 3, 16>(g, st);                                  // three CTAs per SM
}

extern "C" double bta_diag_gemm_flop(int M, int N, int K, int klo, int khi, int out) {
  GemmArgs g{nullptr, nullptr, nullptr, M, N, K, 0, 0, 0, 1.0, 0.0, GEMM_NN, klo, khi, out, nullptr, 0, 0};
  return gemm_alg_flop(g);
}

// Diagnostic: record one {start, end, sm, shape} entry per GEMM CTA into buf[cap][4] (device memory, caller-owned);
// buf = nullptr switches it off.  Not part of the hot path's interface.
extern "C" int bta_debug_cta_trace(unsigned long long* buf, unsigned int cap) {
  const unsigned int zero = 0;
  BTA_CUDA_OK(cudaDeviceSynchronize());
  BTA_CUDA_OK(cudaMemcpyToSymbol(g_cta_trace, &buf, sizeof buf));
  BTA_CUDA_OK(cudaMemcpyToSymbol(g_cta_cap, &cap, sizeof cap));
  BTA_CUDA_OK(cudaMemcpyToSymbol(g_cta_n, &zero, sizeof zero));
  g_trace_host = buf != nullptr;
  return BTA_OK;
}
extern "C" int bta_debug_cta_trace_count(unsigned int* n) {
  if (!n) return BTA_ERR_ARG;
  BTA_CUDA_OK(cudaDeviceSynchronize());
  BTA_CUDA_OK(cudaMemcpyFromSymbol(n, g_cta_n, sizeof *n));
  return BTA_OK;
}
