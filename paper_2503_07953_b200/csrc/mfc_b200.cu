// mfc_b200.cu — kernels and C ABI (include/mfc_b200.h) of the B200-native MFC hot path.
//
// Kernels (all templated on <N fluids, D dimensions>, fp64, SoA x-fastest layout):
//   prim_kernel     pointwise cons->prim (O2)
//   sweep_x         x-direction: one warp per row segment, lane = cell; the warp walks along x in 32-cell
//                   chunks; primitives live in a warp-private shared-memory ring, left face states and
//                   fluxes move between neighbouring lanes by warp shuffles (O1-O5)
//   sweep_march     y/z-direction: lanes span x (coalesced), each thread marches along the sweep
//                   direction with a thread-private 5-cell ring of primitives in shared memory; the
//                   previous face's left state and flux stay in registers (O1-O5)
//   rk_cell         SSP-RK3 stage combination + A10 clamp (O6), applied by the last sweep of each stage
//   cfl_kernel      max_cells sum_d (|u_d|+c)/dx_d by warp shuffles + block reduce + integer atomicMax (O7)
// No face state, flux or primitive array is ever written to HBM; ghost cells are index maps (O1).
#include "../../include/mfc_b200.h"

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "mfc_device.cuh"

namespace mfc {

constexpr unsigned FULL = 0xffffffffu;
// The template parameter WV of the sweeps encodes the nonlinear weights (WV % 3: WENO_JS / WENO_M / WENO_Z) and the
// volume-fraction model (WV / 3: 0 Allaire, 1 Kapila) — both compile-time, so that neither costs the other anything.
#define KAPILA_ON(kp) (WV >= 3)
// Launch shapes (the measured best on B200).
constexpr int XW = 4;      // warps per block, sweep_x
constexpr int XMINB = 3;   // __launch_bounds__ min blocks per SM, sweep_x (168 registers: 12 warps per SM)
constexpr int MB = 128;    // threads per block, sweep_march
constexpr int PB = 256;   // threads per block, pointwise kernels

// ------------------------------------------------------------------------------------------------ prim
template <int N, int D>
__global__ void __launch_bounds__(PB) prim_kernel(const __grid_constant__ KP kp, const double* q, double* w) {  // q, w may alias
  constexpr int NEQ = 2 * N + D + 1;
  const long long c = (long long)blockIdx.x * PB + threadIdx.x;
  if (c >= kp.ncells) return;
  double qc[NEQ], wc[NEQ];
#pragma unroll
  for (int v = 0; v < NEQ; ++v) qc[v] = q[v * kp.ncells + c];
  if (prim_cell<N, D, true>(kp, qc, wc)) *kp.flag = 1;
#pragma unroll
  for (int v = 0; v < NEQ; ++v) w[v * kp.ncells + c] = wc[v];
}

// ------------------------------------------------------------------------------------------------ RK stage of one cell
// O6, each product and sum rounded individually in the printed grouping:
//   stage 1: q1 = q + dt L        stage 2: q2 = 3/4 q + 1/4 (q1 + dt L)        stage 3: q = 1/3 q + 2/3 (q2 + dt L)
// followed by the A10 clamp of the new stage state.  r holds L on entry and the new stage state on exit;
// qn = the cell of q^n, qs = the cell of the stage state the RHS was evaluated on (unused in stage 1).
template <int N, int D, int STAGE>
__device__ __forceinline__ void rk_cell(const KP& kp, double dt, const double* qn, const double* qs, double* r) {
  constexpr int NEQ = 2 * N + D + 1, IA = N + D + 1;
#pragma unroll
  for (int v = 0; v < NEQ; ++v) {
    const double dl = __dmul_rn(dt, r[v]);
    if (STAGE == 1) {
      r[v] = __dadd_rn(qn[v], dl);
    } else if (STAGE == 2) {
      r[v] = __dadd_rn(__dmul_rn(0.75, qn[v]), __dmul_rn(0.25, __dadd_rn(qs[v], dl)));
    } else {
      r[v] = __dadd_rn(__dmul_rn(1.0 / 3.0, qn[v]), __dmul_rn(2.0 / 3.0, __dadd_rn(qs[v], dl)));
    }
  }
  if (kp.clamp) {  // A10
#pragma unroll
    for (int i = 0; i < N; ++i) r[i] = r[i] < 0.0 ? 0.0 : r[i];
    bool marked = false;
#pragma unroll
    for (int i = 0; i < N; ++i)
      if (r[IA + i] < kp.alpha_floor) {
        r[IA + i] = kp.alpha_floor;
        marked = true;
      }
    if (marked) {
      double sum = r[IA];
#pragma unroll
      for (int i = 1; i < N; ++i) sum = __dadd_rn(sum, r[IA + i]);
#pragma unroll
      for (int i = 0; i < N; ++i) r[IA + i] = __ddiv_rn(r[IA + i], sum);
    }
  }
}

// ------------------------------------------------------------------------------------------------ x sweep
// Positions along a segment [s0, s0+L): load position pos <-> cell s0-3+pos (pos = 0..L+5);
// reconstruction position p <-> cell i = s0-1+p (p = 0..L+1), whose stencil sits at load positions p..p+4.
// Lane with position p: reconstructs cell i (both values), solves face i-1/2 (p >= 1) with the left
// state of lane p-1, and updates cell i-1 (p >= 2) with the flux of lane p-1.
// STAGE = 0: rhs = (or +=) the x part of L(q).  STAGE = 1..3 (the last sweep of an RK stage): the
// finished L of the cell goes straight through rk_cell and the new stage state is written instead of L —
// stages 1 and 2 in place over the partial L in `rhs`, stage 3 over q^n in `qnn` (each cell of those buffers is
// read and written by its one thread only; `q`, the state being swept, is never written).
// Work items are (row, segment) pairs, item = row * nseg + segment; a warp owns a contiguous range of items and
// walks through them as ONE stream of positions: the L+6 load positions of an item are followed directly by those of
// the next, so that the two extra reconstruction positions per item cost 2/32 of a warp step instead of a whole
// one (nx = 256: 8.2 steps per row instead of 9).  The grid is one wave of resident blocks (launch_x).
struct XCursor {
  int item, p, s0, nload, rowoff;  // position p of item `item`; s0, nload = L+6, rowoff = row*nx of that item
};

template <int N, int D, bool ACCUM, int STAGE, int WV>
__global__ void __launch_bounds__(XW * 32, XMINB) sweep_x(const __grid_constant__ KP kp, const double* __restrict__ q,
                                                   double* __restrict__ rhs, int seglen, int nseg, double* qnn, double dt,
                                                   int chunk, unsigned* next_chunk, unsigned* reset_other) {
  constexpr int NEQ = 2 * N + D + 1, IA = N + D + 1;
  __shared__ double ring[XW][NEQ][64];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int nx = kp.n[0];
  const long long nitems = kp.ncells / nx * nseg;
  double(*rg)[64] = ring[warp];
  const double idx = kp.inv_dx[0];
  const int lo = kp.bc_lo[0], hi = kp.bc_hi[0];
  bool bad = false;
  const double dtv = (STAGE >= 1 && kp.dt_dev) ? __ldg(kp.dt_dev) : dt;  // mfc_advance keeps dt on the device; read it once
  int it1 = 0;  // end of the current chunk of items

  auto set_item = [&](XCursor& c) {
    const int row = c.item / nseg;
    c.s0 = (c.item - row * nseg) * seglen;
    c.nload = min(seglen, nx - c.s0) + 6;
    c.rowoff = row * nx;
  };
  auto advance = [&](XCursor& c, int by) {
    c.p += by;
    while (c.item < it1 && c.p >= c.nload) {
      c.p -= c.nload;
      ++c.item;
      set_item(c);
    }
  };
  double qn[NEQ];
  auto load = [&](const XCursor& c) {
    if (c.item < it1) {
      int g = c.s0 - 3 + c.p;  // O1: cells -3..nx+2
      if (nx >= 3) {
        if (g < 0) g = lo == BC_PERIODIC ? g + nx : 0;
        if (g >= nx) g = hi == BC_PERIODIC ? g - nx : nx - 1;
      } else {
        g = ghost_index(g, nx, lo, hi);
      }
#pragma unroll
      for (int v = 0; v < NEQ; ++v) qn[v] = __ldg(q + v * kp.ncells + (c.rowoff + g));
    }
  };
  auto store = [&](const XCursor& c, int Q) {
    if (c.item < it1) {
      double w[NEQ];
      bad |= prim_cell<N, D, false>(kp, qn, w);
#pragma unroll
      for (int v = 0; v < NEQ; ++v) rg[v][Q & 63] = w[v];
    }
  };
  // chunks of `chunk` consecutive items are handed out dynamically (one atomic per chunk), so that the warps of the
  // single wave finish together.  Two counters alternate between launches: this launch zeroes the one the next launch
  // on the stream will use (no memset between the sweeps).
  if (blockIdx.x == 0 && threadIdx.x == 0) *reset_other = 0u;
  for (;;) {
  unsigned ck = 0;
  if (lane == 0) ck = atomicAdd(next_chunk, 1u);
  ck = __shfl_sync(FULL, ck, 0);
  if ((long long)ck * chunk >= nitems) break;
  const int it0 = (int)ck * chunk;
  it1 = (int)min((long long)it0 + chunk, nitems);
  XCursor lc;  // load cursor: two chunks ahead of the reconstruction cursor
  lc.item = it0;
  lc.p = 0;
  set_item(lc);
  advance(lc, lane);
  XCursor rc = lc;
  load(lc);
  store(lc, lane);
  advance(lc, 32);
  load(lc);
  store(lc, 32 + lane);
  advance(lc, 32);
  __syncwarp();

  double WLc[NEQ], Fc[NEQ], ufc = 0.0;  // this lane's values of the previous step (lane 31 feeds lane 0)
#pragma unroll
  for (int v = 0; v < NEQ; ++v) WLc[v] = Fc[v] = 0.0;
  const int src = (lane + 31) & 31;
  const bool last = lane == 31;

  for (int Q = lane;; Q += 32) {
    // a lane still has work if it is inside the reconstruction range of the last item or before that item
    const bool more = rc.item < it1 - 1 || (rc.item == it1 - 1 && rc.p < rc.nload - 4);
    if (!__any_sync(FULL, more)) break;
    load(lc);
    const int p = rc.p, nrec = rc.nload - 4;
    const bool act = rc.item < it1 && p < nrec;
    double WL[NEQ], WR[NEQ];
#pragma unroll
    for (int v = 0; v < NEQ; ++v)
      weno5<WV % 3>(rg[v][Q & 63], rg[v][(Q + 1) & 63], rg[v][(Q + 2) & 63], rg[v][(Q + 3) & 63], rg[v][(Q + 4) & 63],
            kp.eps4, WL[v], WR[v]);
    // left neighbour's value by a rotate: lane 31 sends what it had in the previous step
    double WLf[NEQ];
#pragma unroll
    for (int v = 0; v < NEQ; ++v) {
      WLf[v] = __shfl_sync(FULL, last ? WLc[v] : WL[v], src);
      WLc[v] = WL[v];
    }
    double F[NEQ], uf;
    const bool fbad = hllc<N, D, 0>(kp, WLf, WR, F, uf);
    if (act && p >= 1) bad |= fbad;
    double Fm[NEQ], ufm;
#pragma unroll
    for (int v = 0; v < NEQ; ++v) {
      Fm[v] = __shfl_sync(FULL, last ? Fc[v] : F[v], src);
      Fc[v] = F[v];
    }
    ufm = __shfl_sync(FULL, last ? ufc : uf, src);
    ufc = uf;
    if (act && p >= 2) {  // cell i = s0 + p - 2: eq.(10) and the alpha_i div(u) source
      const int off = rc.rowoff + rc.s0 + p - 2;
      const double du = (uf - ufm) * idx;
      double r[NEQ];
#pragma unroll
      for (int v = 0; v < NEQ; ++v) {
        r[v] = (Fm[v] - F[v]) * idx;
        if (v >= IA) r[v] = fma(rg[v][(Q + 1) & 63], du, r[v]);
      }
      if (N == 2 && KAPILA_ON(kp)) {  // K div(u), this direction's part (eq. 5)
        const double Kdu = kapila_K(kp, rg[N + D][(Q + 1) & 63], rg[IA][(Q + 1) & 63], rg[IA + 1][(Q + 1) & 63]) * du;
        r[IA] += Kdu;
        r[IA + 1] -= Kdu;
      }
      if (ACCUM) {
#pragma unroll
        for (int v = 0; v < NEQ; ++v) r[v] += rhs[v * kp.ncells + off];
      }
      if (STAGE >= 1) {
        double qnc[NEQ], qsc[NEQ];
#pragma unroll
        for (int v = 0; v < NEQ; ++v) {
          qnc[v] = qnn[v * kp.ncells + off];
          qsc[v] = STAGE >= 2 ? __ldg(q + v * kp.ncells + off) : 0.0;
        }
        rk_cell<N, D, STAGE>(kp, dtv, qnc, qsc, r);
      }
      double* out = STAGE == 3 ? qnn : rhs;
#pragma unroll
      for (int v = 0; v < NEQ; ++v) out[v * kp.ncells + off] = r[v];
    }
    __syncwarp();
    store(lc, Q + 64);
    advance(lc, 32);
    advance(rc, 32);
    __syncwarp();
  }
  }
  if (bad) *kp.flag = 1;
}

// ------------------------------------------------------------------------------------------------ y/z sweep
// Thread <-> (column, segment [s0, s0+L) along DIR).  Step p = 0..L+1 handles cell g = s0-1+p, whose stencil is
// cells g-2..g+2.  What WENO needs of a cell is formed ONCE, when the cell enters the stencil as cell g+2, and
// carried in thread-private shared-memory rings: its primitives w (3 slots: g-1, g, g+1), its first
// difference d = w - w_prev (3 slots: d1, d2, d3) and u = 13/3 (d - d_prev)^2 + 4 eps (2 slots: u0, u1).  The
// entering cell (g+2) was prefetched as conservatives into registers during the previous step.
// STAGE as in sweep_x.  The operands of the cell update of step p (its partial L, and for STAGE >= 1 its q^n and
// stage-state cells) are fetched by cp.async into thread-private shared-memory slots at the top of the step and
// waited for just before the update, so their latency hides behind the step's arithmetic without holding registers.
__device__ __forceinline__ void cp_async8(double* sdst, const double* gsrc) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(sdst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sa), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
constexpr int MARCH_RING = 8;  // 3 w + 3 d + 2 u slots
// The cell of the stage state (RK stages 2, 3) is staged like the other operands of the update unless that slot would push
// the block over half of the SM's shared memory (NEQ >= 9: 11 slots = 112 KB, one block per SM); then it is read directly
// (it was loaded three steps earlier as cell g+2 of the sweep: an L1/L2 hit).  Config 5: z sweeps 10.7 -> 10.2 ms.
__host__ __device__ constexpr bool march_qs_staged(int neq, int stage) { return stage >= 2 && neq <= 8; }
__host__ __device__ constexpr int march_slots(bool accum, int stage, int neq) {
  return MARCH_RING + (accum ? 1 : 0) + (stage >= 1 ? 1 : 0) + (march_qs_staged(neq, stage) ? 1 : 0);
}

template <int N, int D, int DIR, bool ACCUM, int STAGE, int WV>
__global__ void __launch_bounds__(MB, 1) sweep_march(const __grid_constant__ KP kp, const double* __restrict__ q,
                                                  double* __restrict__ rhs, int seglen, int nseg, double* qnn, double dt) {
  constexpr int NEQ = 2 * N + D + 1, IA = N + D + 1;
  constexpr int NH = (NEQ + 1) / 2;  // variables are stored in pairs (double2) so that every ring access moves two
  constexpr int SLOT = NH * MB;      // double2 per slot
  constexpr int S_D = 3, S_U = 6, S_ACC = MARCH_RING, S_QN = MARCH_RING + (ACCUM ? 1 : 0), S_QS = S_QN + 1;
  extern __shared__ double2 ring[];  // [slots][NH][MB] double2 = variables (2h, 2h+1)
  const int n = kp.n[DIR];
  const int ncols = (int)(kp.ncells / n);
  const long long id = (long long)blockIdx.x * MB + threadIdx.x;
  if (id >= (long long)ncols * nseg) return;
  const int seg = (int)(id / ncols);
  const int col = (int)(id - (long long)seg * ncols);
  // cell offsets within one variable fit 32 bits (mfc_init_grid refuses grids of 2^31 cells or more)
  int base, stride;
  if (DIR == 1) {
    const int nx = kp.n[0];
    const int k = col / nx;
    base = k * nx * kp.n[1] + (col - k * nx);
    stride = nx;
  } else {
    base = col;
    stride = kp.n[0] * kp.n[1];
  }
  const int s0 = seg * seglen;
  const int L = min(seglen, n - s0);
  const int lo = kp.bc_lo[DIR], hi = kp.bc_hi[DIR];
  const double idx = kp.inv_dx[DIR];
  // BF: the prefetch and the cp.async staging are issued unconditionally (on a valid, unused cell outside their range)
  // instead of under a branch.  Measured on B200: 2 % faster for z, 3.5 % slower for y.
  constexpr bool BF = DIR == 2;
  // element (double2 offset o within the ring, pair h): one 16-byte access
  auto ld2 = [&](int o, int h) -> double2 { return ring[o + h * MB + threadIdx.x]; };
  auto st2 = [&](int o, int h, double2 x) { ring[o + h * MB + threadIdx.x] = x; };
  auto elem = [&](int o, int v) -> double* {  // address of variable v in the slot at double2 offset o
    return reinterpret_cast<double*>(ring) + 2 * (o + (v / 2) * MB + threadIdx.x) + (v & 1);
  };
#define RG(slot, v) (*elem((slot) * SLOT, (v)))
  bool bad = false;
  const double dtv = (STAGE >= 1 && kp.dt_dev) ? __ldg(kp.dt_dev) : dt;  // mfc_advance keeps dt on the device; read it once
  double qn[NEQ];
  auto loadq = [&](int off) {
#pragma unroll
    for (int v = 0; v < NEQ; ++v) qn[v] = __ldg(q + v * kp.ncells + off);
  };
  // BC_HALO (last direction only): ghost layer l = 0..2 beyond an end comes from the halo array of that end,
  // [neq][3][plane] with plane == stride; `base` is the column's offset within a plane.
  constexpr bool HALO_DIR = DIR == D - 1;
  auto loadh = [&](const double* halo, int layer) {
    const double* src = halo + ((long long)layer * stride + base);
#pragma unroll
    for (int v = 0; v < NEQ; ++v) qn[v] = __ldg(src + (long long)v * 3 * stride);
  };
  auto load_cell = [&](int cell) {  // logical cell -3..n+2 through the ghost map (O1) or the halo
    if (HALO_DIR && lo == BC_HALO && cell < 0) loadh(kp.halo_lo, cell + 3);
    else if (HALO_DIR && hi == BC_HALO && cell >= n) loadh(kp.halo_hi, min(cell - n, 2));
    else loadq(base + ghost_index(cell, n, lo, hi) * stride);
  };
  // rotating slot offsets (in doubles): i0 = oldest of the 3-slot rings (w of cell g-1, d1), i2 = newest;
  // j0 = older of the 2 u slots.
  int i0 = 0, i1 = SLOT, i2 = 2 * SLOT, j0 = 0, j1 = SLOT;
  {  // prologue: cells s0-3 .. s0 enter one by one (the first differences of the first two are never used)
    double wp[NEQ], dp[NEQ];
#pragma unroll
    for (int v = 0; v < NEQ; ++v) wp[v] = dp[v] = 0.0;
#pragma unroll 1
    for (int m = 0; m < 4; ++m) {
      load_cell(s0 - 3 + m);
      double w[NEQ];
      bad |= prim_cell<N, D, false>(kp, qn, w);
      double dn[2 * NH], un[2 * NH], wn[2 * NH];
#pragma unroll
      for (int v = 0; v < NEQ; ++v) {
        const double d = w[v] - wp[v];
        wn[v] = w[v];
        dn[v] = d;
        un[v] = weno5_u(d - dp[v], kp.eps4);
        wp[v] = w[v];
        dp[v] = d;
      }
      if (NEQ & 1) wn[NEQ] = dn[NEQ] = un[NEQ] = 0.0;
#pragma unroll
      for (int h = 0; h < NH; ++h) {
        st2(i0, h, make_double2(wn[2 * h], wn[2 * h + 1]));
        st2(S_D * SLOT + i0, h, make_double2(dn[2 * h], dn[2 * h + 1]));
        st2(S_U * SLOT + j0, h, make_double2(un[2 * h], un[2 * h + 1]));
      }
      const int t = i0;
      i0 = i1, i1 = i2, i2 = t;
      const int u = j0;
      j0 = j1, j1 = u;
    }
  }
  load_cell(s0 + 1);
  // In the loop the cell to prefetch, s0+2+p, is never below 0, so its ghost map (O1) is: itself below n, else
  // (periodic) itself minus n, reduced once or twice more when n < 3, or (extrapolation) n-1.  Offsets advance
  // by one stride per step.
  int cl = s0 + 2;                          // logical cell to prefetch during step p
  const int nwrap = hi == BC_PERIODIC ? n : 0x7fffffff;  // period of the ghost map at the high end (none: extrapolation clamps)

  double WLp[NEQ], Fp[NEQ], ufp = 0.0;
#pragma unroll
  for (int v = 0; v < NEQ; ++v) WLp[v] = Fp[v] = 0.0;
  int offc = base + (s0 - 2) * stride;      // cell g-1 of step p (used for p >= 2)
#pragma unroll 1
  for (int p = 0; p <= L + 1; ++p) {
    double am[N];  // alpha_i of cell g-1 (source term of its update), read before its slot is reused
#pragma unroll
    for (int i = 0; i < N; ++i) am[i] = *elem(i0, IA + i);
    const double pm = (N == 2 && KAPILA_ON(kp)) ? *elem(i0, N + D) : 0.0;  // its pressure, for K (Kapila model only)
    double w[NEQ];
    bad |= prim_cell<N, D, false>(kp, qn, w);  // cell g+2
    {  // prefetch of cell s0+3+p, branch-free (in the last step, p = L+1, the value is not used; any valid cell will do)
      int gl = cl;
      gl -= gl >= nwrap ? nwrap : 0;
      gl -= gl >= nwrap ? nwrap : 0;
      gl -= gl >= nwrap ? nwrap : 0;
      gl = min(gl, n - 1);
      if (HALO_DIR && hi == BC_HALO && cl >= n) {
        if (BF || p <= L) loadh(kp.halo_hi, min(cl - n, 2));
      } else {
        if (BF || p <= L) loadq(base + gl * stride);
      }
    }
    ++cl;
    if ((ACCUM || STAGE >= 1) && (BF || p >= 2)) {  // operands of this step's update
      // BF, p < 2: nothing is updated yet, but the copies are issued all the same — and they are NOT waited for before step 2
      // issues its own into the same slots.  cp.async groups may land in any order, so the two early copies must carry what
      // step 2's carries: the segment's first cell (offc of step 2).  (They used to read the column's cell 0: when one of them
      // landed last, the first cell of a segment other than the first was updated with the operands of cell 0 — a few times
      // in a thousand steps of config 4 at 128^3; found by the 50-step parity test.)
      const int offs = p >= 2 ? offc : base + s0 * stride;
#pragma unroll
      for (int v = 0; v < NEQ; ++v) {
        if (ACCUM) cp_async8(&RG(S_ACC, v), rhs + v * kp.ncells + offs);
        if (STAGE >= 1) cp_async8(&RG(S_QN, v), qnn + v * kp.ncells + offs);
        if (march_qs_staged(NEQ, STAGE)) cp_async8(&RG(S_QS, v), q + v * kp.ncells + offs);
      }
      cp_async_commit();
    }
    double WL[NEQ], WR[NEQ];
#pragma unroll
    for (int h = 0; h < NH; ++h) {
      const double2 c = ld2(i1, h), dd = ld2(i2, h);
      const double2 d1 = ld2(S_D * SLOT + i0, h), d2 = ld2(S_D * SLOT + i1, h), d3 = ld2(S_D * SLOT + i2, h);
      const double2 u0 = ld2(S_U * SLOT + j0, h), u1 = ld2(S_U * SLOT + j1, h);
      const bool two = 2 * h + 1 < NEQ;
      double2 d4, u2;
      d4.x = w[2 * h] - dd.x;
      u2.x = weno5_u(d4.x - d3.x, kp.eps4);
      d4.y = two ? w[two ? 2 * h + 1 : 0] - dd.y : 0.0;
      u2.y = two ? weno5_u(d4.y - d3.y, kp.eps4) : 0.0;
      st2(i0, h, make_double2(w[2 * h], two ? w[two ? 2 * h + 1 : 0] : 0.0));
      st2(S_D * SLOT + i0, h, d4);
      st2(S_U * SLOT + j0, h, u2);
      weno5_core<WV % 3>(c.x, d1.x, d2.x, d3.x, d4.x, u0.x, u1.x, u2.x, WL[2 * h], WR[2 * h]);
      if (two) weno5_core<WV % 3>(c.y, d1.y, d2.y, d3.y, d4.y, u0.y, u1.y, u2.y, WL[two ? 2 * h + 1 : 0], WR[two ? 2 * h + 1 : 0]);
    }
    {
      const int t = i0;
      i0 = i1, i1 = i2, i2 = t;
      const int u = j0;
      j0 = j1, j1 = u;
    }
    double F[NEQ], uf;
    const bool fbad = hllc<N, D, DIR>(kp, WLp, WR, F, uf);  // face g-1/2: WL of cell g-1, WR of cell g
    bad |= fbad && p >= 1;
    if (p >= 2) {
      const double du = (uf - ufp) * idx;
      double r[NEQ];
#pragma unroll
      for (int v = 0; v < NEQ; ++v) {
        r[v] = (Fp[v] - F[v]) * idx;
        if (v >= IA) r[v] = fma(am[v - IA], du, r[v]);
      }
      if (N == 2 && KAPILA_ON(kp)) {  // K div(u), this direction's part (eq. 5)
        const double Kdu = kapila_K(kp, pm, am[0], am[N - 1]) * du;
        r[IA] += Kdu;
        r[IA + 1] -= Kdu;
      }
      if (ACCUM || STAGE >= 1) cp_async_wait_all();
      if (ACCUM) {
#pragma unroll
        for (int h = 0; h < NH; ++h) {
          const double2 a = ld2(S_ACC * SLOT, h);
          r[2 * h] += a.x;
          if (2 * h + 1 < NEQ) r[2 * h + 1 < NEQ ? 2 * h + 1 : 0] += a.y;
        }
      }
      if (STAGE >= 1) {
        double qnc[NEQ], qsc[NEQ];
#pragma unroll
        for (int h = 0; h < NH; ++h) {
          const double2 a = ld2(S_QN * SLOT, h);
          double2 b = make_double2(0.0, 0.0);
          if (march_qs_staged(NEQ, STAGE)) {
            b = ld2(S_QS * SLOT, h);
          } else if (STAGE >= 2) {
            b.x = __ldg(q + (2 * h) * kp.ncells + offc);
            if (2 * h + 1 < NEQ) b.y = __ldg(q + (2 * h + 1) * kp.ncells + offc);
          }
          qnc[2 * h] = a.x;
          qsc[2 * h] = b.x;
          if (2 * h + 1 < NEQ) {
            qnc[2 * h + 1 < NEQ ? 2 * h + 1 : 0] = a.y;
            qsc[2 * h + 1 < NEQ ? 2 * h + 1 : 0] = b.y;
          }
        }
        rk_cell<N, D, STAGE>(kp, dtv, qnc, qsc, r);
      }
      double* out = STAGE == 3 ? qnn : rhs;
#pragma unroll
      for (int v = 0; v < NEQ; ++v) out[v * kp.ncells + offc] = r[v];
    }
#pragma unroll
    for (int v = 0; v < NEQ; ++v) {
      Fp[v] = F[v];
      WLp[v] = WL[v];
    }
    ufp = uf;
    offc += stride;
  }
#undef RG
  if (bad) *kp.flag = 1;
}

// ------------------------------------------------------------------------------------------------ CFL
// O7 / A9.  All operations IEEE-rounded in the order of the definition, so the per-cell sums — and their
// maximum, which does not depend on the order of comparison — are reproducible bit for bit.
// Positive doubles order like their bit patterns, so the maximum is an integer atomicMax.
template <int N, int D>
__global__ void __launch_bounds__(PB) cfl_kernel(const __grid_constant__ KP kp, const double* __restrict__ q,
                                                 unsigned long long* smax_bits) {
  constexpr int NEQ = 2 * N + D + 1, IM = N, IE = N + D, IA = N + D + 1;
  double smax = 0.0;
  bool bad = false;
  for (long long c = (long long)blockIdx.x * PB + threadIdx.x; c < kp.ncells; c += (long long)gridDim.x * PB) {
    double qc[NEQ], w[NEQ];
#pragma unroll
    for (int v = 0; v < NEQ; ++v) qc[v] = q[v * kp.ncells + c];
    bad |= prim_cell<N, D, true>(kp, qc, w);
    double rho = w[0], Gam = __dmul_rn(w[IA], kp.G[0]), Pi = __dmul_rn(w[IA], kp.P[0]);
#pragma unroll
    for (int i = 1; i < N; ++i) {
      rho = __dadd_rn(rho, w[i]);
      Gam = __dadd_rn(Gam, __dmul_rn(w[IA + i], kp.G[i]));
      Pi = __dadd_rn(Pi, __dmul_rn(w[IA + i], kp.P[i]));
    }
    const double c2 = __ddiv_rn(__dadd_rn(__dmul_rn(__dadd_rn(Gam, 1.0), w[IE]), Pi), __dmul_rn(Gam, rho));
    bad |= !(c2 > 0.0);
    const double cs = __dsqrt_rn(c2);
    double s = __ddiv_rn(__dadd_rn(fabs(w[IM]), cs), kp.dx[0]);
#pragma unroll
    for (int d = 1; d < D; ++d) s = __dadd_rn(s, __ddiv_rn(__dadd_rn(fabs(w[IM + d]), cs), kp.dx[d]));
    smax = s > smax ? s : smax;
  }
#pragma unroll
  for (int o = 16; o; o >>= 1) {
    const double t = __shfl_xor_sync(FULL, smax, o);
    smax = t > smax ? t : smax;
  }
  __shared__ double part[PB / 32];
  if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = smax;
  __syncthreads();
  if (threadIdx.x < 32) {
    smax = threadIdx.x < PB / 32 ? part[threadIdx.x] : 0.0;
#pragma unroll
    for (int o = 16; o; o >>= 1) {
      const double t = __shfl_xor_sync(FULL, smax, o);
      smax = t > smax ? t : smax;
    }
    if (threadIdx.x == 0 && smax > 0.0) atomicMax(smax_bits, (unsigned long long)__double_as_longlong(smax));
  }
  if (bad) *kp.flag = 1;
}

// dt = cfl / (maximum left by cfl_kernel), t += dt, and the maximum is cleared for the next reduction: keeps the time
// step on the device so that mfc_advance needs no host round trip per step.  IEEE operations, the host's arithmetic.
__global__ void dt_kernel(unsigned long long* smax_bits, double cfl, double* dt_t) {
  const double smax = __longlong_as_double((long long)*smax_bits);
  const double dt = __ddiv_rn(cfl, smax);
  dt_t[0] = dt;
  dt_t[1] = __dadd_rn(dt_t[1], dt);
  *smax_bits = 0ull;
}

// ------------------------------------------------------------------------------------------------ unit entry points
template <int WV>
__global__ void __launch_bounds__(PB) weno5_unit_kernel(const __grid_constant__ KP kp, const double* __restrict__ s,
                                                        long long count, double* left, double* right) {
  const long long t = (long long)blockIdx.x * PB + threadIdx.x;
  if (t >= count) return;
  double L, R;
  weno5<WV>(s[5 * t], s[5 * t + 1], s[5 * t + 2], s[5 * t + 3], s[5 * t + 4], kp.eps4, L, R);
  left[t] = L;
  right[t] = R;
}

template <int N, int D, int DIR>
__global__ void __launch_bounds__(PB) hllc_unit_kernel(const __grid_constant__ KP kp, const double* __restrict__ wL,
                                                       const double* __restrict__ wR, long long count, double* F,
                                                       double* uf) {
  constexpr int NEQ = 2 * N + D + 1;
  const long long t = (long long)blockIdx.x * PB + threadIdx.x;
  if (t >= count) return;
  double l[NEQ], r[NEQ], f[NEQ], u;
#pragma unroll
  for (int v = 0; v < NEQ; ++v) {
    l[v] = wL[t * NEQ + v];
    r[v] = wR[t * NEQ + v];
  }
  if (hllc<N, D, DIR>(kp, l, r, f, u)) *kp.flag = 1;
#pragma unroll
  for (int v = 0; v < NEQ; ++v) F[t * NEQ + v] = f[v];
  uf[t] = u;
}

// fsqrt_ratio(a, a b) as the Riemann solver calls it for the face sound speed (a = cn, b = Gamma rho), and the raw
// hardware seed rsqrt(a b) it starts from — so that a test can measure both against the correctly rounded sqrt(a / b).
__global__ void __launch_bounds__(PB) sqrt_ratio_unit_kernel(const double* __restrict__ a, const double* __restrict__ b,
                                                             long long count, double* out, double* seed_out) {
  const long long t = (long long)blockIdx.x * PB + threadIdx.x;
  if (t >= count) return;
  const double ct = a[t] * b[t];
  out[t] = fsqrt_ratio(a[t], ct);
  if (seed_out) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(ct));
    seed_out[t] = y;
  }
}

// ------------------------------------------------------------------------------------------------ viscous terms
// O8 (eqs.(1),(2); reading A22): T = 2 eta (D - tr(D) I/3) with one uniform eta, second-order
// central differences at face centres.  Two pointwise kernels, bound by HBM/L2, run BEFORE the sweeps of an RHS evaluation:
// velocity_kernel writes u_d = (rho u_d)/rho, viscous_kernel overwrites rhs with the viscous rates of momentum and
// energy (zero for the other equations); the x sweep then accumulates onto it.
template <int N, int D>
__global__ void __launch_bounds__(PB) velocity_kernel(const __grid_constant__ KP kp, const double* __restrict__ q,
                                                      double* __restrict__ vel) {
  const long long c = (long long)blockIdx.x * PB + threadIdx.x;
  if (c >= kp.ncells) return;
  double rho = q[c];
#pragma unroll
  for (int i = 1; i < N; ++i) rho = __dadd_rn(rho, q[i * kp.ncells + c]);
#pragma unroll
  for (int d = 0; d < D; ++d) vel[d * kp.ncells + c] = __ddiv_rn(q[(N + d) * kp.ncells + c], rho);
}

// the same for the ghost layer next to each end of the last direction that takes its ghost cells from a halo array
// (layer 2 of halo_lo = cell -1, layer 0 of halo_hi = cell n; halo layout [neq][3][plane])
template <int N, int D>
__global__ void __launch_bounds__(PB) velocity_halo_kernel(const __grid_constant__ KP kp, double* vel_lo, double* vel_hi) {
  const long long plane = kp.ncells / kp.n[D - 1];
  const long long c = (long long)blockIdx.x * PB + threadIdx.x;
  if (c >= plane) return;
#pragma unroll
  for (int end = 0; end < 2; ++end) {
    const double* h = end ? kp.halo_hi : kp.halo_lo;
    double* out = end ? vel_hi : vel_lo;
    if (!h || (end ? kp.bc_hi[D - 1] : kp.bc_lo[D - 1]) != BC_HALO) continue;
    const int layer = end ? 0 : 2;
    double rho = h[(0 * 3 + layer) * plane + c];
#pragma unroll
    for (int i = 1; i < N; ++i) rho = __dadd_rn(rho, h[(i * 3 + layer) * plane + c]);
#pragma unroll
    for (int d = 0; d < D; ++d) out[d * plane + c] = __ddiv_rn(h[((N + d) * 3 + layer) * plane + c], rho);
  }
}

template <int N, int D>
__global__ void __launch_bounds__(PB) viscous_kernel(const __grid_constant__ KP kp, const double* __restrict__ vel,
                                                     double* __restrict__ rhs) {
  constexpr int NEQ = 2 * N + D + 1;
  const long long c = (long long)blockIdx.x * PB + threadIdx.x;
  if (c >= kp.ncells) return;
  const int nx = kp.n[0], ny = kp.n[1];
  int ijk[3];
  ijk[0] = (int)(c % nx);
  ijk[1] = (int)((c / nx) % ny);
  ijk[2] = (int)(c / ((long long)nx * ny));
  // mapped neighbour indices per direction (O1): nb[d][o+1], o = -1, 0, +1 (the generic map only where n < 3)
  int nb[3][3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    const int n = kp.n[d], i = ijk[d];
    nb[d][1] = i;
    if (d < D && n >= 3) {
      nb[d][0] = i > 0 ? i - 1 : (kp.bc_lo[d] == BC_PERIODIC ? n - 1 : 0);
      nb[d][2] = i < n - 1 ? i + 1 : (kp.bc_hi[d] == BC_PERIODIC ? 0 : n - 1);
    } else {
      nb[d][0] = d < D ? ghost_index(i - 1, n, kp.bc_lo[d], kp.bc_hi[d]) : 0;
      nb[d][2] = d < D ? ghost_index(i + 1, n, kp.bc_lo[d], kp.bc_hi[d]) : 0;
    }
  }
  // the three layers of the last direction: base of component 0 and the stride between components — the interior array, or
  // (MFC_BC_HALO: a slab end) the ghost layer's velocities
  constexpr int LD = D - 1;
  const int plane = (int)(kp.ncells / kp.n[LD]);  // cells of one layer of the last direction
  const double* lbase[3];
  long long lstride[3];
#pragma unroll
  for (int o = 0; o < 3; ++o) {
    lbase[o] = vel + (long long)nb[LD][o] * plane;
    lstride[o] = kp.ncells;
  }
  if (D >= 2 && ijk[LD] == 0 && kp.bc_lo[LD] == BC_HALO) lbase[0] = kp.vel_halo_lo, lstride[0] = plane;
  if (D >= 2 && ijk[LD] == kp.n[LD] - 1 && kp.bc_hi[LD] == BC_HALO) lbase[2] = kp.vel_halo_hi, lstride[2] = plane;
  int rowoff[3];  // D = 3: offset of row j' within a layer, 32-bit (fewer than 2^31 cells)
#pragma unroll
  for (int oy = 0; oy < 3; ++oy) rowoff[oy] = D == 3 ? nb[1][oy] * nx : 0;
  auto U = [&](int m, const int* o) {  // velocity component m at offset o[3] from the cell
    const int ol = o[LD] + 1;
    const int inplane = D == 1 ? 0 : (D == 3 ? rowoff[o[1] + 1] : 0) + nb[0][o[0] + 1];
    return __ldg(lbase[ol] + m * lstride[ol] + inplane);
  };
  double acc[D + 1];
#pragma unroll
  for (int m = 0; m <= D; ++m) acc[m] = 0.0;
#pragma unroll
  for (int d = 0; d < D; ++d) {
#pragma unroll
    for (int side = 0; side < 2; ++side) {  // side 1: face between the cell and its upper neighbour; 0: lower neighbour and the cell
      int a[3] = {0, 0, 0}, b[3] = {0, 0, 0};
      a[d] = side - 1;
      b[d] = side;
      double grad[D][D], uf[D];
#pragma unroll
      for (int m = 0; m < D; ++m) {
        const double ua = U(m, a), ub = U(m, b);
        uf[m] = 0.5 * (ua + ub);
#pragma unroll
        for (int e = 0; e < D; ++e) {
          if (e == d) {
            grad[m][e] = (ub - ua) * kp.inv_dx[d];
          } else {
            int ap[3] = {a[0], a[1], a[2]}, am[3] = {a[0], a[1], a[2]}, bp[3] = {b[0], b[1], b[2]}, bm[3] = {b[0], b[1], b[2]};
            ap[e] += 1, am[e] -= 1, bp[e] += 1, bm[e] -= 1;
            grad[m][e] = 0.25 * kp.inv_dx[e] * ((U(m, ap) - U(m, am)) + (U(m, bp) - U(m, bm)));
          }
        }
      }
      double div = 0.0;
#pragma unroll
      for (int m = 0; m < D; ++m) div += grad[m][m];
      const double sgn = side ? kp.inv_dx[d] : -kp.inv_dx[d];
      double G = 0.0;
#pragma unroll
      for (int m = 0; m < D; ++m) {
        double T = kp.eta * (grad[m][d] + grad[d][m]);
        if (m == d) T = fma(-(2.0 / 3.0) * kp.eta, div, T);
        G = fma(T, uf[m], G);
        acc[m] = fma(sgn, T, acc[m]);
      }
      acc[D] = fma(sgn, G, acc[D]);
    }
  }
#pragma unroll
  for (int v = 0; v < NEQ; ++v) {
    double r = 0.0;
    if (v >= N && v < N + D) r = acc[v - N];
    if (v == N + D) r = acc[D];
    rhs[v * kp.ncells + c] = r;
  }
}

// ------------------------------------------------------------------------------------------------ FP64 peak probe
// DFMA chains on registers, 8 independent chains per thread, 16 warps per SM (mfc_measure_fp64).
// MODE 0: x = fma(x, a, b) with loop-invariant a, b — the pipe's issue rate.  MODE 1: x_i = fma(x_i, x_j, x_k) with three
// distinct, changing register operands — what an FP64 instruction costs when it reads three different registers.
template <int MODE>
__global__ void __launch_bounds__(128) dfma_probe_kernel(double* out, int iters, double a, double b) {
  double x[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) x[i] = 1.0 + 1e-3 * threadIdx.x + i;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
      for (int i = 0; i < 8; ++i) x[i] = MODE == 0 ? fma(x[i], a, b) : fma(x[i], x[(i + 1) & 7], x[(i + 3) & 7]);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += x[i];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace mfc

// ================================================================================================ host side
using namespace mfc;

struct mfc_grid {
  KP kp;
  int ndim, nf, neq;
  int weno = 0;  // WENO_JS / WENO_M / WENO_Z
  int device;
  cudaStream_t stream;
  double* q1 = nullptr;     // stage state
  double* Lq = nullptr;     // rhs scratch
  double* vel = nullptr;    // velocities u_d (D arrays), only when eta > 0
  double* vel_halo = nullptr;  // with MFC_BC_HALO: velocities of the ghost layer next to each end, [2][D][plane]
  double* hq = nullptr;     // device staging for the *_host calls (lazy)
  double* hr = nullptr;
  unsigned long long* d_red = nullptr;  // [0] = smax bits
  int* d_flag = nullptr;
  double* d_dt = nullptr;               // [0] dt of the step in flight, [1] elapsed time (mfc_advance)
  unsigned* d_xnext = nullptr;          // two work counters of sweep_x, used alternately (each launch zeroes the other)
  int xparity = 0;
  unsigned long long* h_red = nullptr;  // pinned: [0] smax bits, [1] flag
  int seg[3];
  long long launches = 0;
  // CUDA graph of two mfc_advance steps for launch-bound grids (advance_pairs_graph)
  bool step_graph = true;               // mfc_set_step_graph
  bool adv_warm = false;                // two plain steps have run on this handle (every launch function has done its one-time queries)
  cudaGraphExec_t adv_exec = nullptr;
  const double* adv_q = nullptr;        // what the instantiated graph was captured for
  double adv_cfl = 0.0;
  int adv_parity = 0;
  long long adv_kernels = 0;            // kernels in the graph
  cudaStream_t gstream = nullptr;       // capture / replay stream (the handle's own may be the legacy stream, which cannot capture)
  cudaEvent_t gev_in = nullptr, gev_out = nullptr;
  int num_sms = 148;
  // per-kernel device timing (mfc_set_profiling)
  bool profiling = false;
  struct Rec { int cls; cudaEvent_t a, b; };
  std::vector<Rec> recs;
  std::vector<cudaEvent_t> pool;
  double prof_ms[MFC_K_COUNT] = {};
  long long prof_n[MFC_K_COUNT] = {};
};

// Brackets one launch with events when profiling is on; always counts the launch.
struct Scope {
  mfc_grid* g;
  cudaEvent_t b = nullptr;
  Scope(mfc_grid* g_, int cls);
  ~Scope();
};

static thread_local std::string g_err;
static mfc_status fail(mfc_status s, const std::string& m) {
  g_err = m;
  return s;
}
static mfc_status cuda_fail(cudaError_t e, const char* what) {
  return fail(MFC_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
#define CK(call)                                       \
  do {                                                 \
    cudaError_t e_ = (call);                           \
    if (e_ != cudaSuccess) return cuda_fail(e_, #call); \
  } while (0)

static cudaEvent_t get_event(mfc_grid* g) {
  if (!g->pool.empty()) {
    cudaEvent_t e = g->pool.back();
    g->pool.pop_back();
    return e;
  }
  cudaEvent_t e = nullptr;
  cudaEventCreate(&e);
  return e;
}
Scope::Scope(mfc_grid* g_, int cls) : g(g_) {
  g->launches++;
  if (g->profiling) {
    cudaEvent_t a = get_event(g);
    b = get_event(g);
    cudaEventRecord(a, g->stream);
    g->recs.push_back({cls, a, b});
  }
}
Scope::~Scope() {
  if (b) cudaEventRecord(b, g->stream);
}
// fold finished records into the per-class sums (caller has synchronised the stream)
static void drain_profile(mfc_grid* g) {
  for (auto& r : g->recs) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, r.a, r.b) == cudaSuccess) {
      g->prof_ms[r.cls] += ms;
      g->prof_n[r.cls]++;
    }
    g->pool.push_back(r.a);
    g->pool.push_back(r.b);
  }
  g->recs.clear();
}

// MFC_BC_HALO: which ends of the last direction take their ghost layers from the halo arrays
static bool halo_lo_on(const mfc_grid* g) { return g->kp.bc_lo[g->ndim - 1] == BC_HALO; }
static bool halo_hi_on(const mfc_grid* g) { return g->kp.bc_hi[g->ndim - 1] == BC_HALO; }
static bool halo_missing(const mfc_grid* g) {
  return (halo_lo_on(g) && !g->kp.halo_lo) || (halo_hi_on(g) && !g->kp.halo_hi);
}

static size_t state_bytes(const mfc_grid* g) { return sizeof(double) * (size_t)g->neq * (size_t)g->kp.ncells; }

// segment lengths: long enough that the halo work (2 extra reconstructions, 6 extra conversions per
// segment) is small, short enough that every SM gets several blocks.
static void default_segments(mfc_grid* g) {
  const long long cells = g->kp.ncells;
  {  // x: warps = rows * nseg; a segment of L cells needs ceil((L+2)/32) warp steps -> L = 32k - 2
    const int nx = g->kp.n[0];
    const long long rows = cells / nx;
    const long long want_warps = (long long)g->num_sms * 32;
    int L = nx;
    if (rows < want_warps) {
      const long long nseg = (want_warps + rows - 1) / rows;
      long long l = (nx + nseg - 1) / nseg;
      l = ((l + 2 + 31) / 32) * 32 - 2;
      if (l < 30) l = 30;
      if (l < nx) L = (int)l;
    }
    g->seg[0] = L;
  }
  for (int d = 1; d < g->ndim; ++d) {
    const int n = g->kp.n[d];
    const long long cols = cells / n;
    const long long want_threads = (long long)g->num_sms * 1536;
    int L = n;
    if (cols < want_threads) {
      const long long nseg = (want_threads + cols - 1) / cols;
      long long l = (n + nseg - 1) / nseg;
      if (l < 8) l = 8;
      // short segments pay 2 extra reconstructions and a 4-cell prologue each: take 32 cells if that still fills
      // three quarters of the resident threads (2 blocks of MB per SM), measured on config 3: 8 % faster than 8
      if (l < 32 && n >= 32 && cols * ((n + 31) / 32) * 4 >= (long long)g->num_sms * 2 * MB * 3) l = 32;
      if (l < n) L = (int)l;
    }
    g->seg[d] = L;
  }
}

template <int N, int D>
static cudaError_t launch_prim(mfc_grid* g, const double* q, double* w) {
  const long long nb = (g->kp.ncells + PB - 1) / PB;
  Scope sc(g, MFC_K_PRIM);
  prim_kernel<N, D><<<(unsigned)nb, PB, 0, g->stream>>>(g->kp, q, w);
  return cudaGetLastError();
}

template <int N, int D, int WV, int DIR, bool ACCUM, int STAGE>
static cudaError_t launch_march(mfc_grid* g, const double* q, double* rhs, double* qn, double dt) {
  if constexpr (DIR < D) {
    constexpr int NEQ = 2 * N + D + 1;
    const int n = g->kp.n[DIR];
    const int seglen = g->seg[DIR];
    const int nseg = (n + seglen - 1) / seglen;
    const long long threads = g->kp.ncells / n * nseg;
    const long long nb = (threads + MB - 1) / MB;
    const size_t smem = sizeof(double2) * march_slots(ACCUM, STAGE, NEQ) * ((NEQ + 1) / 2) * MB;
    auto kern = sweep_march<N, D, DIR, ACCUM, STAGE, WV>;
    static bool attr_done[16] = {};
    if (!attr_done[g->device & 15]) {
      cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      if (e != cudaSuccess) return e;
      attr_done[g->device & 15] = true;
    }
    Scope sc(g, DIR == 1 ? MFC_K_SWEEP_Y : MFC_K_SWEEP_Z);
    kern<<<(unsigned)nb, MB, smem, g->stream>>>(g->kp, q, rhs, seglen, nseg, qn, dt);
    return cudaGetLastError();
  } else {
    return cudaSuccess;
  }
}

template <int N, int D, int WV, bool ACCUM, int STAGE>
static cudaError_t launch_x(mfc_grid* g, const double* q, double* rhs, double* qn, double dt) {
  const int nx = g->kp.n[0];
  const int seglen = g->seg[0];
  const int nseg = (nx + seglen - 1) / seglen;
  const long long items = g->kp.ncells / nx * nseg;
  auto kern = sweep_x<N, D, ACCUM, STAGE, WV>;
  static int resident[16] = {};  // blocks per SM of this instantiation, per device
  int& res = resident[g->device & 15];
  if (res == 0) {
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&res, kern, XW * 32, 0);
    if (e != cudaSuccess) return e;
    if (res < 1) res = 1;
  }
  // one wave of resident blocks; the warps take chunks of consecutive items from a counter until none is left
  long long nb = (items + XW - 1) / XW;
  const long long wave = (long long)res * g->num_sms;
  if (nb > wave) nb = wave;
  // chunk: about 8 chunks per warp for balance, at least 1 item, at most 16 (longer streams gain nothing)
  long long chunk = items / (nb * XW * 8);
  if (chunk < 1) chunk = 1;
  if (chunk > 16) chunk = 16;
  unsigned* cur = g->d_xnext + (g->xparity & 1);
  unsigned* other = g->d_xnext + ((g->xparity + 1) & 1);
  g->xparity ^= 1;
  Scope sc(g, MFC_K_SWEEP_X);
  kern<<<(unsigned)nb, XW * 32, 0, g->stream>>>(g->kp, q, rhs, seglen, nseg, qn, dt, (int)chunk, cur, other);
  return cudaGetLastError();
}

// viscous rates of momentum and energy written over rhs (zero elsewhere); the x sweep accumulates onto them
template <int N, int D>
static cudaError_t launch_viscous(mfc_grid* g, const double* q, double* rhs) {
  const unsigned nb = (unsigned)((g->kp.ncells + PB - 1) / PB);
  {
    Scope sc(g, MFC_K_PRIM);
    velocity_kernel<N, D><<<nb, PB, 0, g->stream>>>(g->kp, q, g->vel);
  }
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  if (g->vel_halo) {  // slab ends: the velocities of the ghost layer from the halo arrays
    if constexpr (D >= 2) {
      const long long plane = g->kp.ncells / g->kp.n[D - 1];
      Scope sc(g, MFC_K_PRIM);
      velocity_halo_kernel<N, D><<<(unsigned)((plane + PB - 1) / PB), PB, 0, g->stream>>>(
          g->kp, g->vel_halo, g->vel_halo + (size_t)D * plane);
      if ((e = cudaGetLastError()) != cudaSuccess) return e;
    }
  }
  Scope sc(g, MFC_K_PRIM);
  viscous_kernel<N, D><<<nb, PB, 0, g->stream>>>(g->kp, g->vel, rhs);
  return cudaGetLastError();
}

// rhs = L(q) restricted to the directions in mask.  mask == all: x overwrites, y and z accumulate.
template <int N, int D, int WV>
static cudaError_t launch_rhs(mfc_grid* g, const double* q, double* rhs, int mask) {
  if constexpr (WV >= 3 && N != 2) return cudaErrorInvalidValue;  // Kapila: two fluids only (not instantiated otherwise)
  else {
  const int all = (1 << D) - 1;
  cudaError_t e;
  if (mask == 7 && g->kp.eta > 0.0) {  // the viscous rates belong to the whole RHS only (dir_mask == 7, as in mfc_rhs)
    if ((e = launch_viscous<N, D>(g, q, rhs)) != cudaSuccess) return e;
    if ((e = launch_x<N, D, WV, true, 0>(g, q, rhs, nullptr, 0.0)) != cudaSuccess) return e;
  } else if ((mask & all) == all) {
    if ((e = launch_x<N, D, WV, false, 0>(g, q, rhs, nullptr, 0.0)) != cudaSuccess) return e;
  } else {
    if ((e = cudaMemsetAsync(rhs, 0, state_bytes(g), g->stream)) != cudaSuccess) return e;
    if (mask & 1)
      if ((e = launch_x<N, D, WV, true, 0>(g, q, rhs, nullptr, 0.0)) != cudaSuccess) return e;
  }
  if (D >= 2 && (mask & 2))
    if ((e = launch_march<N, D, WV, 1, true, 0>(g, q, rhs, nullptr, 0.0)) != cudaSuccess) return e;
  if (D >= 3 && (mask & 4))
    if ((e = launch_march<N, D, WV, 2, true, 0>(g, q, rhs, nullptr, 0.0)) != cudaSuccess) return e;
  return cudaSuccess;
  }
}

// One RK stage: L(qs) by the D sweeps, the last of which applies the stage combination and the clamp itself
// (no separate RK kernel, the finished L never goes to HBM).  Stages 1 and 2 leave the new stage state in `work`
// (where the partial L was), stage 3 writes q^{n+1} over q^n.
// parts: bit 0 = the sweeps that do not touch the last direction (they need no halo of a slab), bit 1 = the last sweep,
// which also applies the RK stage.  3 = the whole stage.
template <int N, int D, int WV, int STAGE>
static cudaError_t launch_stage(mfc_grid* g, const double* qs, double* work, double* qn, double dt, int parts = 3) {
  cudaError_t e;
  const bool visc = g->kp.eta > 0.0;
  if constexpr (D == 1) {
    if (!(parts & 2)) return cudaSuccess;
    if (visc)
      if ((e = launch_viscous<N, D>(g, qs, work)) != cudaSuccess) return e;
    return visc ? launch_x<N, D, WV, true, STAGE>(g, qs, work, qn, dt) : launch_x<N, D, WV, false, STAGE>(g, qs, work, qn, dt);
  } else {
    // on a slab the viscous stencil reads the ghost layer of the last direction: nothing of the stage can start before the halos
    // have landed, so part 1 is empty and part 2 is the whole stage
    if (visc && (halo_lo_on(g) || halo_hi_on(g))) {
      if (!(parts & 2)) return cudaSuccess;
      parts = 3;
    }
    if (parts & 1) {
      if (visc)
        if ((e = launch_viscous<N, D>(g, qs, work)) != cudaSuccess) return e;
      e = visc ? launch_x<N, D, WV, true, 0>(g, qs, work, nullptr, 0.0) : launch_x<N, D, WV, false, 0>(g, qs, work, nullptr, 0.0);
      if (e != cudaSuccess) return e;
      if constexpr (D == 3)
        if ((e = launch_march<N, D, WV, 1, true, 0>(g, qs, work, nullptr, 0.0)) != cudaSuccess) return e;
    }
    if (!(parts & 2)) return cudaSuccess;
    if constexpr (D == 2) {
      return launch_march<N, D, WV, 1, true, STAGE>(g, qs, work, qn, dt);
    } else {
      return launch_march<N, D, WV, 2, true, STAGE>(g, qs, work, qn, dt);
    }
  }
}

// O6: q^n in `q` (caller's), two work arrays A = Lq, B = q1:
//   stage 1 sweeps q,  partial L in A, q1 ends in A;   stage 2 sweeps A, partial L in B, q2 ends in B;
//   stage 3 sweeps B,  partial L in A, q^{n+1} ends in q.
template <int N, int D, int WV>
static cudaError_t launch_rk3(mfc_grid* g, double* q, double dt) {
  if constexpr (WV >= 3 && N != 2) return cudaErrorInvalidValue;  // Kapila: two fluids only
  else {
    cudaError_t e;
    if ((e = launch_stage<N, D, WV, 1>(g, q, g->Lq, q, dt)) != cudaSuccess) return e;
    if ((e = launch_stage<N, D, WV, 2>(g, g->Lq, g->q1, q, dt)) != cudaSuccess) return e;
    return launch_stage<N, D, WV, 3>(g, g->q1, g->Lq, q, dt);
  }
}

template <int N, int D>
static cudaError_t launch_hllc_unit(mfc_grid* g, int dir, const double* wL, const double* wR, long long count, double* F,
                                    double* uf) {
  const long long nb = (count + PB - 1) / PB;
  Scope sc(g, MFC_K_PRIM);
  if (dir == 0) hllc_unit_kernel<N, D, 0><<<(unsigned)nb, PB, 0, g->stream>>>(g->kp, wL, wR, count, F, uf);
  if constexpr (D >= 2)
    if (dir == 1) hllc_unit_kernel<N, D, 1><<<(unsigned)nb, PB, 0, g->stream>>>(g->kp, wL, wR, count, F, uf);
  if constexpr (D >= 3)
    if (dir == 2) hllc_unit_kernel<N, D, 2><<<(unsigned)nb, PB, 0, g->stream>>>(g->kp, wL, wR, count, F, uf);
  return cudaGetLastError();
}

template <int N, int D>
static cudaError_t launch_cfl(mfc_grid* g, const double* q) {
  long long nb = (g->kp.ncells + PB - 1) / PB;
  const long long cap = (long long)g->num_sms * 8;
  if (nb > cap) nb = cap;
  Scope sc(g, MFC_K_CFL);
  cfl_kernel<N, D><<<(unsigned)nb, PB, 0, g->stream>>>(g->kp, q, g->d_red);
  return cudaGetLastError();
}

#define MFC_DISPATCH(g, EXPR)                                  \
  [&]() -> cudaError_t {                                       \
    switch ((g)->nf * 10 + (g)->ndim) {                        \
      case 11: { constexpr int N = 1, D = 1; return EXPR; }    \
      case 12: { constexpr int N = 1, D = 2; return EXPR; }    \
      case 13: { constexpr int N = 1, D = 3; return EXPR; }    \
      case 21: { constexpr int N = 2, D = 1; return EXPR; }    \
      case 22: { constexpr int N = 2, D = 2; return EXPR; }    \
      case 23: { constexpr int N = 2, D = 3; return EXPR; }    \
      case 31: { constexpr int N = 3, D = 1; return EXPR; }    \
      case 32: { constexpr int N = 3, D = 2; return EXPR; }    \
      case 33: { constexpr int N = 3, D = 3; return EXPR; }    \
    }                                                          \
    return cudaErrorInvalidValue;                              \
  }()

// the same with the weights variant WV of the handle as a third compile-time constant
#define MFC_DISPATCH_W1(g, K, EXPR)                                                          \
  switch ((g)->weno) {                                                                           \
    case WENO_JS: { constexpr int WV = WENO_JS + 3 * K; return MFC_DISPATCH(g, EXPR); }          \
    case WENO_M: { constexpr int WV = WENO_M + 3 * K; return MFC_DISPATCH(g, EXPR); }            \
    case WENO_Z: { constexpr int WV = WENO_Z + 3 * K; return MFC_DISPATCH(g, EXPR); }            \
  }
#define MFC_DISPATCH_W(g, EXPR)                                                                  \
  [&]() -> cudaError_t {                                                                         \
    if ((g)->kp.kapila) {                                                                        \
      MFC_DISPATCH_W1(g, 1, EXPR)                                                                \
    } else {                                                                                     \
      MFC_DISPATCH_W1(g, 0, EXPR)                                                                \
    }                                                                                            \
    return cudaErrorInvalidValue;                                                                \
  }()

template <int N, int D, int WV>
static cudaError_t launch_rk3_stage(mfc_grid* g, double* q, double dt, int stage, int parts) {
  if constexpr (WV >= 3 && N != 2) return cudaErrorInvalidValue;
  else {
    if (stage == 1) return launch_stage<N, D, WV, 1>(g, q, g->Lq, q, dt, parts);
    if (stage == 2) return launch_stage<N, D, WV, 2>(g, g->Lq, g->q1, q, dt, parts);
    return launch_stage<N, D, WV, 3>(g, g->q1, g->Lq, q, dt, parts);
  }
}


static void drop_step_graph(mfc_grid* g) {
  if (g->adv_exec) cudaGraphExecDestroy(g->adv_exec);
  g->adv_exec = nullptr;
}

static mfc_status use_device(const mfc_grid* g) {
  CK(cudaSetDevice(g->device));
  return MFC_OK;
}

extern "C" {

const char* mfc_last_error(void) { return g_err.c_str(); }

mfc_status mfc_init_grid(const mfc_params* p, mfc_grid** out) {
  if (!p || !out) return fail(MFC_ERR_ARG, "mfc_init_grid: NULL argument");
  *out = nullptr;
  if (p->ndim < 1 || p->ndim > 3) return fail(MFC_ERR_ARG, "mfc_init_grid: ndim must be 1..3");
  if (p->nfluids < 1 || p->nfluids > MFC_MAX_FLUIDS) return fail(MFC_ERR_ARG, "mfc_init_grid: nfluids must be 1..3");
  if (!p->gamma || !p->pi_inf) return fail(MFC_ERR_ARG, "mfc_init_grid: gamma/pi_inf NULL");
  long long cells = 1;
  for (int d = 0; d < 3; ++d) {
    if (p->n[d] < 1) return fail(MFC_ERR_ARG, "mfc_init_grid: n[d] must be >= 1");
    if (d >= p->ndim && p->n[d] != 1) return fail(MFC_ERR_ARG, "mfc_init_grid: n[d] must be 1 for d >= ndim");
    if (d < p->ndim && !(p->dx[d] > 0.0)) return fail(MFC_ERR_ARG, "mfc_init_grid: dx[d] must be > 0");
    const bool halo_ok = p->ndim >= 2 && d == p->ndim - 1;  // MFC_BC_HALO: last direction of a 2-D / 3-D grid only
    if (p->bc_lo[d] != MFC_BC_PERIODIC && p->bc_lo[d] != MFC_BC_EXTRAP && !(halo_ok && p->bc_lo[d] == MFC_BC_HALO))
      return fail(MFC_ERR_ARG, "mfc_init_grid: bad bc_lo");
    if (p->bc_hi[d] != MFC_BC_PERIODIC && p->bc_hi[d] != MFC_BC_EXTRAP && !(halo_ok && p->bc_hi[d] == MFC_BC_HALO))
      return fail(MFC_ERR_ARG, "mfc_init_grid: bad bc_hi");
    if ((p->bc_lo[d] == MFC_BC_PERIODIC) != (p->bc_hi[d] == MFC_BC_PERIODIC))
      return fail(MFC_ERR_ARG, "mfc_init_grid: periodic must be set on both ends of a direction");
    cells *= p->n[d];
    if (cells >= (1LL << 31)) return fail(MFC_ERR_ARG, "mfc_init_grid: grid too large (cell offsets are 32-bit: fewer than 2^31 cells)");
  }
  for (int i = 0; i < p->nfluids; ++i)
    if (!(p->gamma[i] > 1.0)) return fail(MFC_ERR_ARG, "mfc_init_grid: gamma_i must be > 1");
  if (!(p->weno_eps > 0.0)) return fail(MFC_ERR_ARG, "mfc_init_grid: weno_eps must be > 0");
  // the weights are evaluated in product form: (4 eps)^4 must not underflow where all three indicators vanish
  if (p->weno_eps < 1e-75) return fail(MFC_ERR_ARG, "mfc_init_grid: weno_eps must be >= 1e-75 (product form of the weights)");
  if (p->model != MFC_MODEL_ALLAIRE && p->model != MFC_MODEL_KAPILA)
    return fail(MFC_ERR_ARG, "mfc_init_grid: model must be MFC_MODEL_ALLAIRE or MFC_MODEL_KAPILA");
  if (p->model == MFC_MODEL_KAPILA && p->nfluids != 2)
    return fail(MFC_ERR_ARG, "mfc_init_grid: MFC_MODEL_KAPILA is defined for two fluids (PAPER.md:78, eq. 5)");
  if (!(p->eta >= 0.0)) return fail(MFC_ERR_ARG, "mfc_init_grid: eta must be >= 0");
  if (p->weno != MFC_WENO_JS && p->weno != MFC_WENO_M && p->weno != MFC_WENO_Z)
    return fail(MFC_ERR_ARG, "mfc_init_grid: weno must be MFC_WENO_JS, MFC_WENO_M or MFC_WENO_Z");
  int ndev = 0;
  CK(cudaGetDeviceCount(&ndev));
  if (p->device < 0 || p->device >= ndev) return fail(MFC_ERR_ARG, "mfc_init_grid: no such CUDA device");
  CK(cudaSetDevice(p->device));

  mfc_grid* g = new (std::nothrow) mfc_grid();
  if (!g) return fail(MFC_ERR_ALLOC, "mfc_init_grid: out of host memory");
  std::memset(&g->kp, 0, sizeof(KP));
  g->ndim = p->ndim;
  g->nf = p->nfluids;
  g->weno = p->weno;
  g->neq = 2 * p->nfluids + p->ndim + 1;
  g->device = p->device;
  g->stream = (cudaStream_t)p->stream;
  for (int d = 0; d < 3; ++d) {
    g->kp.n[d] = p->n[d];
    g->kp.bc_lo[d] = p->bc_lo[d];
    g->kp.bc_hi[d] = p->bc_hi[d];
    g->kp.dx[d] = d < p->ndim ? p->dx[d] : 1.0;
    g->kp.inv_dx[d] = 1.0 / g->kp.dx[d];
  }
  g->kp.ncells = cells;
  for (int i = 0; i < 3; ++i) g->kp.G[i] = g->kp.P[i] = 0.0;
  for (int i = 0; i < p->nfluids; ++i) {  // PAPER.md:117 with eq.(4): rho e = sum alpha_i (p + gamma_i pi_inf_i)/(gamma_i-1)
    g->kp.G[i] = 1.0 / (p->gamma[i] - 1.0);
    g->kp.P[i] = (p->gamma[i] * p->pi_inf[i]) / (p->gamma[i] - 1.0);
  }
  g->kp.eps4 = 4.0 * p->weno_eps;
  g->kp.alpha_floor = p->alpha_floor;
  g->kp.clamp = p->clamp ? 1 : 0;
  g->kp.kapila = p->model == MFC_MODEL_KAPILA ? 1 : 0;
  g->kp.eta = p->eta;
  for (int i = 0; i < 2 && i < p->nfluids; ++i) {
    g->kp.gam[i] = p->gamma[i];
    g->kp.gpi[i] = p->gamma[i] * p->pi_inf[i];
  }
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, p->device) == cudaSuccess) g->num_sms = prop.multiProcessorCount;
  default_segments(g);

  const size_t bytes = state_bytes(g);
  cudaError_t e;
  if ((e = cudaMalloc(&g->q1, bytes)) != cudaSuccess || (e = cudaMalloc(&g->Lq, bytes)) != cudaSuccess ||
      (e = cudaMalloc(&g->d_red, 16)) != cudaSuccess || (e = cudaMalloc(&g->d_flag, sizeof(int))) != cudaSuccess ||
      (e = cudaMalloc(&g->d_dt, 2 * sizeof(double))) != cudaSuccess ||
      (e = cudaMalloc(&g->d_xnext, 2 * sizeof(unsigned))) != cudaSuccess ||
      (e = cudaMallocHost(&g->h_red, 16)) != cudaSuccess) {
    mfc_free_grid(g);
    g_err = std::string("mfc_init_grid: allocation failed: ") + cudaGetErrorString(e);
    cudaGetLastError();
    return MFC_ERR_ALLOC;
  }
  if (g->kp.eta > 0.0 && cudaMalloc(&g->vel, sizeof(double) * (size_t)g->ndim * (size_t)cells) != cudaSuccess) {
    cudaGetLastError();
    mfc_free_grid(g);
    return fail(MFC_ERR_ALLOC, "mfc_init_grid: allocation of the velocity arrays failed");
  }
  if (g->kp.eta > 0.0 && (halo_lo_on(g) || halo_hi_on(g))) {
    const size_t plane = (size_t)(cells / p->n[p->ndim - 1]);
    if (cudaMalloc(&g->vel_halo, sizeof(double) * 2 * (size_t)g->ndim * plane) != cudaSuccess) {
      cudaGetLastError();
      mfc_free_grid(g);
      return fail(MFC_ERR_ALLOC, "mfc_init_grid: allocation of the halo velocities failed");
    }
    g->kp.vel_halo_lo = g->vel_halo;
    g->kp.vel_halo_hi = g->vel_halo + (size_t)g->ndim * plane;
  }
  g->kp.flag = g->d_flag;
  CK(cudaMemsetAsync(g->d_flag, 0, sizeof(int), g->stream));
  CK(cudaMemsetAsync(g->d_red, 0, 16, g->stream));
  CK(cudaMemsetAsync(g->d_xnext, 0, 2 * sizeof(unsigned), g->stream));
  *out = g;
  return MFC_OK;
}

mfc_status mfc_free_grid(mfc_grid* g) {
  if (!g) return MFC_OK;
  cudaSetDevice(g->device);
  cudaStreamSynchronize(g->stream);
  cudaFree(g->q1);
  cudaFree(g->Lq);
  cudaFree(g->vel);
  cudaFree(g->vel_halo);
  cudaFree(g->hq);
  cudaFree(g->hr);
  cudaFree(g->d_red);
  cudaFree(g->d_flag);
  cudaFree(g->d_dt);
  cudaFree(g->d_xnext);
  if (g->h_red) cudaFreeHost(g->h_red);
  drop_step_graph(g);
  if (g->gstream) {
    cudaStreamSynchronize(g->gstream);
    cudaStreamDestroy(g->gstream);
    cudaEventDestroy(g->gev_in);
    cudaEventDestroy(g->gev_out);
  }
  drain_profile(g);
  for (cudaEvent_t e : g->pool) cudaEventDestroy(e);
  delete g;
  return MFC_OK;
}

int mfc_num_eqns(const mfc_grid* g) { return g ? g->neq : -1; }
long long mfc_num_cells(const mfc_grid* g) { return g ? g->kp.ncells : -1; }
long long mfc_launch_count(const mfc_grid* g) { return g ? g->launches : -1; }

mfc_status mfc_set_segments(mfc_grid* g, int seg_x, int seg_y, int seg_z) {
  if (!g) return fail(MFC_ERR_ARG, "mfc_set_segments: NULL handle");
  if (seg_x < 0 || seg_y < 0 || seg_z < 0) return fail(MFC_ERR_ARG, "mfc_set_segments: negative length");
  const int s[3] = {seg_x, seg_y, seg_z};
  mfc_grid tmp = *g;
  default_segments(&tmp);
  for (int d = 0; d < 3; ++d) g->seg[d] = s[d] > 0 ? (s[d] < g->kp.n[d] ? s[d] : g->kp.n[d]) : tmp.seg[d];
  drop_step_graph(g);  // the launch shapes are part of a captured step
  return MFC_OK;
}

mfc_status mfc_set_step_graph(mfc_grid* g, int on) {
  if (!g) return fail(MFC_ERR_ARG, "mfc_set_step_graph: NULL handle");
  g->step_graph = on != 0;
  if (!on) drop_step_graph(g);
  return MFC_OK;
}

mfc_status mfc_prim_from_cons(mfc_grid* g, const double* q, double* w) {
  if (!g || !q || !w) return fail(MFC_ERR_ARG, "mfc_prim_from_cons: NULL argument");
  if (mfc_status s = use_device(g)) return s;
  CK(MFC_DISPATCH(g, (launch_prim<N, D>(g, q, w))));
  return MFC_OK;
}

mfc_status mfc_rhs_dirs(mfc_grid* g, const double* q, double* rhs, int dir_mask) {
  if (!g || !q || !rhs) return fail(MFC_ERR_ARG, "mfc_rhs: NULL argument");
  if (q == rhs) return fail(MFC_ERR_ARG, "mfc_rhs: q and rhs must not alias");
  if (dir_mask < 1 || dir_mask > 7) return fail(MFC_ERR_ARG, "mfc_rhs_dirs: dir_mask must be 1..7 (bit d = direction d)");
  // the viscous rates belong to the whole RHS, which is spelt 7 whatever the number of dimensions: a mask that names all of
  // this grid's directions in another way (3 on a 2-D grid) would silently come back inviscid — refuse it instead
  if (g->kp.eta > 0.0 && dir_mask != 7 && (dir_mask & ((1 << g->ndim) - 1)) == (1 << g->ndim) - 1)
    return fail(MFC_ERR_ARG, "mfc_rhs_dirs: with eta > 0 the full RHS (viscous rates included) is dir_mask 7; a partial mask must leave a direction of the grid out");
  if (halo_missing(g)) return fail(MFC_ERR_ARG, "mfc_rhs: MFC_BC_HALO without mfc_set_halo");
  if (mfc_status s = use_device(g)) return s;
  CK(MFC_DISPATCH_W(g, (launch_rhs<N, D, WV>(g, q, rhs, dir_mask))));
  return MFC_OK;
}

mfc_status mfc_rhs(mfc_grid* g, const double* q, double* rhs) { return mfc_rhs_dirs(g, q, rhs, 7); }

mfc_status mfc_rk3_steps(mfc_grid* g, double* q, double dt, int nsteps) {
  if (!g || !q) return fail(MFC_ERR_ARG, "mfc_rk3_step: NULL argument");
  if (nsteps < 0) return fail(MFC_ERR_ARG, "mfc_rk3_steps: nsteps < 0");
  if (!(dt == dt)) return fail(MFC_ERR_ARG, "mfc_rk3_step: dt is NaN");
  if (halo_lo_on(g) || halo_hi_on(g))
    return fail(MFC_ERR_ARG, "mfc_rk3_step: with MFC_BC_HALO the halos must be refreshed before every stage: use mfc_rk3_stage");
  if (mfc_status s = use_device(g)) return s;
  for (int s = 0; s < nsteps; ++s) CK(MFC_DISPATCH_W(g, (launch_rk3<N, D, WV>(g, q, dt))));
  return MFC_OK;
}

mfc_status mfc_rk3_stage_parts(mfc_grid* g, double* q, double dt, int stage, int parts) {
  if (!g || !q) return fail(MFC_ERR_ARG, "mfc_rk3_stage: NULL argument");
  if (stage < 1 || stage > 3) return fail(MFC_ERR_ARG, "mfc_rk3_stage: stage must be 1, 2 or 3");
  if (parts < 1 || parts > 3) return fail(MFC_ERR_ARG, "mfc_rk3_stage_parts: parts must be 1, 2 or 3");
  if (!(dt == dt)) return fail(MFC_ERR_ARG, "mfc_rk3_stage: dt is NaN");
  if ((parts & 2) && halo_missing(g)) return fail(MFC_ERR_ARG, "mfc_rk3_stage: MFC_BC_HALO without mfc_set_halo");
  if (mfc_status s = use_device(g)) return s;
  CK(MFC_DISPATCH_W(g, (launch_rk3_stage<N, D, WV>(g, q, dt, stage, parts))));
  return MFC_OK;
}

mfc_status mfc_rk3_stage(mfc_grid* g, double* q, double dt, int stage) { return mfc_rk3_stage_parts(g, q, dt, stage, 3); }

mfc_status mfc_stage_input(mfc_grid* g, const double* q, int stage, const double** state_out) {
  if (!g || !q || !state_out) return fail(MFC_ERR_ARG, "mfc_stage_input: NULL argument");
  if (stage < 1 || stage > 3) return fail(MFC_ERR_ARG, "mfc_stage_input: stage must be 1, 2 or 3");
  *state_out = stage == 1 ? q : stage == 2 ? g->Lq : g->q1;
  return MFC_OK;
}

mfc_status mfc_pack_halo(mfc_grid* g, const double* q, int stage, double* send_lo, double* send_hi) {
  if (!g || !q || (!send_lo && !send_hi)) return fail(MFC_ERR_ARG, "mfc_pack_halo: NULL argument");
  if (stage < 1 || stage > 3) return fail(MFC_ERR_ARG, "mfc_pack_halo: stage must be 1, 2 or 3");
  const int nl = g->kp.n[g->ndim - 1];
  if (g->ndim < 2 || nl < 3) return fail(MFC_ERR_ARG, "mfc_pack_halo: needs a 2-D or 3-D grid with at least 3 cells in the last direction");
  if (mfc_status s = use_device(g)) return s;
  const double* st = stage == 1 ? q : stage == 2 ? g->Lq : g->q1;
  const size_t plane = (size_t)(g->kp.ncells / nl);
  const size_t row = 3 * plane * sizeof(double), pitch = (size_t)g->kp.ncells * sizeof(double);
  // per variable the three layers next to an end are contiguous: one strided copy per end
  if (send_lo) CK(cudaMemcpy2DAsync(send_lo, row, st, pitch, row, g->neq, cudaMemcpyDeviceToDevice, g->stream));
  if (send_hi)
    CK(cudaMemcpy2DAsync(send_hi, row, st + (size_t)(nl - 3) * plane, pitch, row, g->neq, cudaMemcpyDeviceToDevice, g->stream));
  return MFC_OK;
}

mfc_status mfc_set_halo(mfc_grid* g, const double* halo_lo, const double* halo_hi) {
  if (!g) return fail(MFC_ERR_ARG, "mfc_set_halo: NULL handle");
  if ((halo_lo_on(g) && !halo_lo) || (halo_hi_on(g) && !halo_hi))
    return fail(MFC_ERR_ARG, "mfc_set_halo: NULL array for an end with MFC_BC_HALO");
  g->kp.halo_lo = halo_lo;
  g->kp.halo_hi = halo_hi;
  return MFC_OK;
}

mfc_status mfc_rk3_step(mfc_grid* g, double* q, double dt) { return mfc_rk3_steps(g, q, dt, 1); }

static mfc_status read_flag_and_sync(mfc_grid* g, bool with_red) {
  CK(cudaMemcpyAsync(&g->h_red[1], g->d_flag, sizeof(int), cudaMemcpyDeviceToHost, g->stream));
  if (with_red) CK(cudaMemcpyAsync(&g->h_red[0], g->d_red, 8, cudaMemcpyDeviceToHost, g->stream));
  CK(cudaMemsetAsync(g->d_flag, 0, sizeof(int), g->stream));
  CK(cudaStreamSynchronize(g->stream));
  if ((int)(g->h_red[1] & 0xffffffffu) != 0) return fail(MFC_ERR_NONPHYSICAL, "non-physical state (rho <= 0 or c^2 <= 0 or NaN)");
  return MFC_OK;
}

mfc_status mfc_cfl_dt(mfc_grid* g, const double* q, double cfl, double* dt_out) {
  if (!g || !q || !dt_out) return fail(MFC_ERR_ARG, "mfc_cfl_dt: NULL argument");
  if (mfc_status s = use_device(g)) return s;
  CK(cudaMemsetAsync(g->d_red, 0, 8, g->stream));
  CK(MFC_DISPATCH(g, (launch_cfl<N, D>(g, q))));
  g->h_red[1] = 0;
  const mfc_status s = read_flag_and_sync(g, true);
  double smax;
  std::memcpy(&smax, &g->h_red[0], 8);
  *dt_out = cfl / smax;
  return s;
}

mfc_status mfc_check(mfc_grid* g) {
  if (!g) return fail(MFC_ERR_ARG, "mfc_check: NULL handle");
  if (mfc_status s = use_device(g)) return s;
  g->h_red[1] = 0;
  return read_flag_and_sync(g, false);
}

static mfc_status ensure_staging(mfc_grid* g, bool need_r) {
  if (!g->hq) {
    if (cudaMalloc(&g->hq, state_bytes(g)) != cudaSuccess) {
      cudaGetLastError();
      return fail(MFC_ERR_ALLOC, "staging allocation failed");
    }
  }
  if (need_r && !g->hr) {
    if (cudaMalloc(&g->hr, state_bytes(g)) != cudaSuccess) {
      cudaGetLastError();
      return fail(MFC_ERR_ALLOC, "staging allocation failed");
    }
  }
  return MFC_OK;
}

mfc_status mfc_rhs_host(mfc_grid* g, const double* q_host, double* rhs_host) {
  if (!g || !q_host || !rhs_host) return fail(MFC_ERR_ARG, "mfc_rhs_host: NULL argument");
  if (halo_missing(g)) return fail(MFC_ERR_ARG, "mfc_rhs_host: MFC_BC_HALO without mfc_set_halo");
  if (mfc_status s = use_device(g)) return s;
  if (mfc_status s = ensure_staging(g, true)) return s;
  CK(cudaMemcpyAsync(g->hq, q_host, state_bytes(g), cudaMemcpyHostToDevice, g->stream));
  CK(MFC_DISPATCH_W(g, (launch_rhs<N, D, WV>(g, g->hq, g->hr, 7))));
  CK(cudaMemcpyAsync(rhs_host, g->hr, state_bytes(g), cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  return MFC_OK;
}

mfc_status mfc_rk3_steps_host(mfc_grid* g, double* q_host, double dt, int nsteps) {
  if (!g || !q_host) return fail(MFC_ERR_ARG, "mfc_rk3_steps_host: NULL argument");
  if (nsteps < 0) return fail(MFC_ERR_ARG, "mfc_rk3_steps_host: nsteps < 0");
  if (halo_lo_on(g) || halo_hi_on(g)) return fail(MFC_ERR_ARG, "mfc_rk3_steps_host: not available with MFC_BC_HALO");
  if (mfc_status s = use_device(g)) return s;
  if (mfc_status s = ensure_staging(g, false)) return s;
  CK(cudaMemcpyAsync(g->hq, q_host, state_bytes(g), cudaMemcpyHostToDevice, g->stream));
  for (int s = 0; s < nsteps; ++s) CK(MFC_DISPATCH_W(g, (launch_rk3<N, D, WV>(g, g->hq, dt))));
  CK(cudaMemcpyAsync(q_host, g->hq, state_bytes(g), cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  return MFC_OK;
}

// CFL + RK3 per step, all on the device: the reduction leaves max_cells sum_d (|u_d|+c)/dx_d, dt_kernel turns it into dt
// and adds it to the elapsed time, the RK stages read dt from device memory.  One host synchronisation at the end, which
// also reports the sticky non-physical flag.  Same kernels and arithmetic as the caller's loop of mfc_cfl_dt + mfc_rk3_step.
static mfc_status advance_steps_plain(mfc_grid* g, double* q, double cfl, int nsteps) {
  for (int s = 0; s < nsteps; ++s) {
    CK(MFC_DISPATCH(g, (launch_cfl<N, D>(g, q))));
    {
      Scope sc(g, MFC_K_CFL);
      dt_kernel<<<1, 1, 0, g->stream>>>(g->d_red, cfl, g->d_dt);
    }
    CK(cudaGetLastError());
    g->kp.dt_dev = g->d_dt;
    const cudaError_t e = MFC_DISPATCH_W(g, (launch_rk3<N, D, WV>(g, q, 0.0)));
    g->kp.dt_dev = nullptr;
    CK(e);
  }
  return MFC_OK;
}

// Launch-bound grids (BASELINE.json configs 1 and 2: 1000 and 4000 cells, 11 launches of a few microseconds each per step):
// the launches of TWO steps are captured once into a CUDA graph and replayed, one graph launch per pair of steps.  Two, not
// one: sweep_x alternates between two work counters from launch to launch (launch_x) and a step has three x sweeps, so only
// after two steps does the next launch find the counters as the capture did.  The graph holds the very kernels, arguments
// and order of advance_steps_plain — same bits — and is re-captured when q, cfl or the counter parity differ from the capture's.
// The handle's stream may be the legacy default stream, which cannot be captured: capture and replay run on a stream of the
// handle's own, ordered against the handle's stream by events on both sides.
constexpr long long STEP_GRAPH_MAX_CELLS = 1 << 18;

static mfc_status advance_pairs_graph(mfc_grid* g, double* q, double cfl, int npairs) {
  if (!g->gstream) {
    CK(cudaStreamCreateWithFlags(&g->gstream, cudaStreamNonBlocking));
    CK(cudaEventCreateWithFlags(&g->gev_in, cudaEventDisableTiming));
    CK(cudaEventCreateWithFlags(&g->gev_out, cudaEventDisableTiming));
  }
  if (!g->adv_exec || g->adv_q != q || g->adv_cfl != cfl || g->adv_parity != g->xparity) {
    drop_step_graph(g);
    const cudaStream_t user = g->stream;
    const long long l0 = g->launches;
    const int parity = g->xparity;
    cudaError_t e = cudaStreamBeginCapture(g->gstream, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) return cuda_fail(e, "cudaStreamBeginCapture");
    g->stream = g->gstream;
    const mfc_status st = advance_steps_plain(g, q, cfl, 2);
    g->stream = user;
    cudaGraph_t graph = nullptr;
    e = cudaStreamEndCapture(g->gstream, &graph);
    g->adv_kernels = g->launches - l0;
    g->launches = l0;          // captured, not run
    g->xparity = parity;       // two steps: an even number of x sweeps, the parity is where it was
    if (st != MFC_OK || e != cudaSuccess) {
      if (graph) cudaGraphDestroy(graph);
      return st != MFC_OK ? st : cuda_fail(e, "cudaStreamEndCapture");
    }
    e = cudaGraphInstantiate(&g->adv_exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) {
      g->adv_exec = nullptr;
      return cuda_fail(e, "cudaGraphInstantiate");
    }
    g->adv_q = q;
    g->adv_cfl = cfl;
    g->adv_parity = parity;
  }
  CK(cudaEventRecord(g->gev_in, g->stream));
  CK(cudaStreamWaitEvent(g->gstream, g->gev_in, 0));
  for (int i = 0; i < npairs; ++i) {
    CK(cudaGraphLaunch(g->adv_exec, g->gstream));
    g->launches += g->adv_kernels;
  }
  CK(cudaEventRecord(g->gev_out, g->gstream));
  CK(cudaStreamWaitEvent(g->stream, g->gev_out, 0));
  return MFC_OK;
}

static mfc_status advance_impl(mfc_grid* g, double* q, double cfl, int nsteps, double* t_out) {
  CK(cudaMemsetAsync(g->d_dt, 0, 2 * sizeof(double), g->stream));
  CK(cudaMemsetAsync(g->d_red, 0, 8, g->stream));
  int left = nsteps;
  if (g->step_graph && !g->profiling && g->kp.ncells <= STEP_GRAPH_MAX_CELLS) {
    if (!g->adv_warm && left >= 2) {  // the first two steps of a handle run plainly (one-time occupancy queries are not captured)
      if (mfc_status s = advance_steps_plain(g, q, cfl, 2)) return s;
      g->adv_warm = true;
      left -= 2;
    }
    if (g->adv_warm && left >= 2) {
      if (mfc_status s = advance_pairs_graph(g, q, cfl, left / 2)) return s;
      left &= 1;
    }
  }
  if (mfc_status s = advance_steps_plain(g, q, cfl, left)) return s;
  CK(cudaMemcpyAsync(&g->h_red[0], g->d_dt + 1, 8, cudaMemcpyDeviceToHost, g->stream));
  g->h_red[1] = 0;
  const mfc_status st = read_flag_and_sync(g, false);
  if (t_out) std::memcpy(t_out, &g->h_red[0], 8);
  return st;
}

mfc_status mfc_advance(mfc_grid* g, double* q, double cfl, int nsteps, double* t_elapsed_host) {
  if (!g || !q) return fail(MFC_ERR_ARG, "mfc_advance: NULL argument");
  if (nsteps < 0 || !(cfl > 0.0)) return fail(MFC_ERR_ARG, "mfc_advance: nsteps < 0 or cfl <= 0");
  if (halo_lo_on(g) || halo_hi_on(g)) return fail(MFC_ERR_ARG, "mfc_advance: not available with MFC_BC_HALO (use mfc_rk3_stage)");
  if (mfc_status s = use_device(g)) return s;
  return advance_impl(g, q, cfl, nsteps, t_elapsed_host);
}

mfc_status mfc_advance_host(mfc_grid* g, double* q_host, double cfl, int nsteps, double* t_elapsed_host) {
  if (!g || !q_host) return fail(MFC_ERR_ARG, "mfc_advance_host: NULL argument");
  if (nsteps < 0 || !(cfl > 0.0)) return fail(MFC_ERR_ARG, "mfc_advance_host: nsteps < 0 or cfl <= 0");
  if (halo_lo_on(g) || halo_hi_on(g)) return fail(MFC_ERR_ARG, "mfc_advance_host: not available with MFC_BC_HALO");
  if (mfc_status s = use_device(g)) return s;
  if (mfc_status s = ensure_staging(g, false)) return s;
  CK(cudaMemcpyAsync(g->hq, q_host, state_bytes(g), cudaMemcpyHostToDevice, g->stream));
  if (mfc_status s = advance_impl(g, g->hq, cfl, nsteps, t_elapsed_host)) return s;
  CK(cudaMemcpyAsync(q_host, g->hq, state_bytes(g), cudaMemcpyDeviceToHost, g->stream));
  CK(cudaStreamSynchronize(g->stream));
  return MFC_OK;
}

mfc_status mfc_weno5_values(mfc_grid* g, const double* stencils, long long count, double* left, double* right) {
  if (!g || !stencils || !left || !right) return fail(MFC_ERR_ARG, "mfc_weno5_values: NULL argument");
  if (count < 0) return fail(MFC_ERR_ARG, "mfc_weno5_values: count < 0");
  if (mfc_status s = use_device(g)) return s;
  if (count == 0) return MFC_OK;
  {
    Scope sc(g, MFC_K_PRIM);
    const unsigned nb = (unsigned)((count + PB - 1) / PB);
    if (g->weno == WENO_M) weno5_unit_kernel<WENO_M><<<nb, PB, 0, g->stream>>>(g->kp, stencils, count, left, right);
    else if (g->weno == WENO_Z) weno5_unit_kernel<WENO_Z><<<nb, PB, 0, g->stream>>>(g->kp, stencils, count, left, right);
    else weno5_unit_kernel<WENO_JS><<<nb, PB, 0, g->stream>>>(g->kp, stencils, count, left, right);
  }
  CK(cudaGetLastError());
  return MFC_OK;
}

mfc_status mfc_hllc_faces(mfc_grid* g, int dir, const double* wL, const double* wR, long long count, double* F, double* uf) {
  if (!g || !wL || !wR || !F || !uf) return fail(MFC_ERR_ARG, "mfc_hllc_faces: NULL argument");
  if (count < 0 || dir < 0 || dir >= g->ndim) return fail(MFC_ERR_ARG, "mfc_hllc_faces: bad count or direction");
  if (mfc_status s = use_device(g)) return s;
  if (count == 0) return MFC_OK;
  CK(MFC_DISPATCH(g, (launch_hllc_unit<N, D>(g, dir, wL, wR, count, F, uf))));
  return MFC_OK;
}

mfc_status mfc_sqrt_ratio_values(mfc_grid* g, const double* a, const double* b, long long count, double* out, double* seed_out) {
  if (!g || !a || !b || !out) return fail(MFC_ERR_ARG, "mfc_sqrt_ratio_values: NULL argument");
  if (count < 0) return fail(MFC_ERR_ARG, "mfc_sqrt_ratio_values: count < 0");
  if (count == 0) return MFC_OK;
  if (mfc_status s = use_device(g)) return s;
  {
    Scope sc(g, MFC_K_PRIM);
    sqrt_ratio_unit_kernel<<<(unsigned)((count + PB - 1) / PB), PB, 0, g->stream>>>(a, b, count, out, seed_out);
  }
  CK(cudaGetLastError());
  return MFC_OK;
}

mfc_status mfc_measure_fp64(int device, void* stream, double* dfma_tflops_host, double* dfma3_tflops_host) {
  if (!dfma_tflops_host || !dfma3_tflops_host) return fail(MFC_ERR_ARG, "mfc_measure_fp64: NULL argument");
  int ndev = 0;
  CK(cudaGetDeviceCount(&ndev));
  if (device < 0 || device >= ndev) return fail(MFC_ERR_ARG, "mfc_measure_fp64: no such CUDA device");
  CK(cudaSetDevice(device));
  cudaDeviceProp prop;
  CK(cudaGetDeviceProperties(&prop, device));
  cudaStream_t st = (cudaStream_t)stream;
  const int blocks = prop.multiProcessorCount * 4, iters = 40000;  // 4 blocks of 128 threads per SM, ~10 ms per launch
  double* out = nullptr;
  CK(cudaMalloc(&out, sizeof(double) * (size_t)blocks * 128));
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  double res[2] = {0.0, 0.0};
  cudaError_t err = cudaSuccess;
  for (int mode = 0; mode < 2 && err == cudaSuccess; ++mode) {
    for (int rep = 0; rep < 3; ++rep) {  // first repetition warms up; best of the other two
      cudaEventRecord(e0, st);
      if (mode == 0) dfma_probe_kernel<0><<<blocks, 128, 0, st>>>(out, iters, 1.0000001, 1e-9);
      else dfma_probe_kernel<1><<<blocks, 128, 0, st>>>(out, iters, 1.0000001, 1e-9);
      cudaEventRecord(e1, st);
      if ((err = cudaEventSynchronize(e1)) != cudaSuccess) break;
      float ms = 0.f;
      cudaEventElapsedTime(&ms, e0, e1);
      const double tf = 2.0 * 32.0 * iters * (double)blocks * 128.0 / (ms * 1e-3) / 1e12;  // 32 DFMA per thread per iteration
      if (rep > 0 && tf > res[mode]) res[mode] = tf;
    }
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(out);
  if (err != cudaSuccess) return cuda_fail(err, "mfc_measure_fp64");
  *dfma_tflops_host = res[0];
  *dfma3_tflops_host = res[1];
  return MFC_OK;
}

mfc_status mfc_set_profiling(mfc_grid* g, int on) {
  if (!g) return fail(MFC_ERR_ARG, "mfc_set_profiling: NULL handle");
  if (mfc_status s = use_device(g)) return s;
  CK(cudaStreamSynchronize(g->stream));
  drain_profile(g);
  if (on) {
    for (int c = 0; c < MFC_K_COUNT; ++c) {
      g->prof_ms[c] = 0.0;
      g->prof_n[c] = 0;
    }
  }
  g->profiling = on != 0;
  return MFC_OK;
}

mfc_status mfc_get_profile(mfc_grid* g, int kernel_class, double* total_ms_host, long long* launches_host) {
  if (!g || !total_ms_host || !launches_host) return fail(MFC_ERR_ARG, "mfc_get_profile: NULL argument");
  if (kernel_class < 0 || kernel_class >= MFC_K_COUNT) return fail(MFC_ERR_ARG, "mfc_get_profile: bad kernel class");
  if (mfc_status s = use_device(g)) return s;
  CK(cudaStreamSynchronize(g->stream));
  drain_profile(g);
  *total_ms_host = g->prof_ms[kernel_class];
  *launches_host = g->prof_n[kernel_class];
  return MFC_OK;
}

}  // extern "C"

// ================================================================================================ mfc_cfl_dt_static
// The CFL reduction for callers that cannot allocate (include/mfc_b200.h: an application whose memory pool owns all of
// HBM, a latency-critical loop, a host that forbids allocation after start-up).  Everything the kernel needs beyond
// its inputs and outputs — one partial maximum per block, the completion counter, the non-physical flag — sits in the
// file-scope array below, which is part of the library image: MFC_STATIC_SCRATCH_BYTES on every GPU that loads the
// library, until the process exits.  No handle, no cudaMalloc / cudaFree / cudaMallocHost on this path.
//
// `static_scratch` as written in HOST code is only the host-side shadow of the device array; handing that to a kernel
// or to cudaMemsetAsync would fault (or, where the GPU can reach host memory, scribble over the shadow).  The host
// therefore asks the runtime for the device address once per device (static_scratch_on) and passes that pointer.
namespace mfc {

constexpr int ST_CPB = MFC_STATIC_CELLS_PER_BLOCK;   // cells reduced by one block
constexpr int ST_MAXB = MFC_STATIC_MAX_BLOCKS;       // partial maxima the array has room for
constexpr int ST_HDR = 1024;                         // bytes in front of the partials: word 0 = blocks finished, word 1 = flag
static_assert(ST_CPB % PB == 0, "a block's cells are dealt to its threads in whole rounds");
static_assert(MFC_STATIC_SCRATCH_BYTES == ST_HDR + 8 * ST_MAXB, "header + one double per block");
static __device__ __align__(256) unsigned char static_scratch[MFC_STATIC_SCRATCH_BYTES];

// Same per-cell arithmetic as cfl_kernel (O7 / A9, every operation IEEE-rounded in the order of the definition), so the
// maximum — which does not depend on the order of comparison — has the same bits.  What differs is where the partial
// results go: block b stores its maximum in part[b]; the block that finishes last (counter in hdr[0]) takes the maximum
// of the gridDim.x partials, writes dt and the flag to the caller's outputs and puts the counter and flag back to zero.
template <int N, int D>
__global__ void __launch_bounds__(PB) cfl_static_kernel(const __grid_constant__ KP kp, const double* __restrict__ q,
                                                        double cfl, unsigned char* scratch, double* dt_out,
                                                        int* nonphysical_out) {
  constexpr int NEQ = 2 * N + D + 1, IM = N, IE = N + D, IA = N + D + 1;
  unsigned* hdr = reinterpret_cast<unsigned*>(scratch);
  double* part = reinterpret_cast<double*>(scratch + ST_HDR);
  double smax = 0.0;
  bool bad = false;
  const long long c0 = (long long)blockIdx.x * ST_CPB + threadIdx.x;
#pragma unroll 2
  for (int k = 0; k < ST_CPB / PB; ++k) {
    const long long c = c0 + (long long)k * PB;
    if (c >= kp.ncells) break;
    double qc[NEQ], w[NEQ];
#pragma unroll
    for (int v = 0; v < NEQ; ++v) qc[v] = q[v * kp.ncells + c];
    bad |= prim_cell<N, D, true>(kp, qc, w);
    double rho = w[0], Gam = __dmul_rn(w[IA], kp.G[0]), Pi = __dmul_rn(w[IA], kp.P[0]);
#pragma unroll
    for (int i = 1; i < N; ++i) {
      rho = __dadd_rn(rho, w[i]);
      Gam = __dadd_rn(Gam, __dmul_rn(w[IA + i], kp.G[i]));
      Pi = __dadd_rn(Pi, __dmul_rn(w[IA + i], kp.P[i]));
    }
    const double c2 = __ddiv_rn(__dadd_rn(__dmul_rn(__dadd_rn(Gam, 1.0), w[IE]), Pi), __dmul_rn(Gam, rho));
    bad |= !(c2 > 0.0);
    const double cs = __dsqrt_rn(c2);
    double s = __ddiv_rn(__dadd_rn(fabs(w[IM]), cs), kp.dx[0]);
#pragma unroll
    for (int d = 1; d < D; ++d) s = __dadd_rn(s, __ddiv_rn(__dadd_rn(fabs(w[IM + d]), cs), kp.dx[d]));
    smax = s > smax ? s : smax;
  }
  __shared__ double wmax[PB / 32];
  __shared__ bool last;
  auto block_max = [&](double x) {  // maximum over the block, valid in thread 0
#pragma unroll
    for (int o = 16; o; o >>= 1) {
      const double t = __shfl_xor_sync(FULL, x, o);
      x = t > x ? t : x;
    }
    if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = x;
    __syncthreads();
    if (threadIdx.x < 32) {
      x = threadIdx.x < PB / 32 ? wmax[threadIdx.x] : 0.0;
#pragma unroll
      for (int o = 16; o; o >>= 1) {
        const double t = __shfl_xor_sync(FULL, x, o);
        x = t > x ? t : x;
      }
    }
    return x;
  };
  smax = block_max(smax);
  const int any_bad = __syncthreads_or(bad ? 1 : 0);
  if (threadIdx.x == 0) {
    part[blockIdx.x] = smax;
    if (any_bad) atomicOr(&hdr[1], 1u);
    __threadfence();  // the partial and the flag are visible before the counter moves
    last = atomicAdd(&hdr[0], 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  double m = 0.0;
  for (unsigned b = threadIdx.x; b < gridDim.x; b += PB) {
    const double t = __ldcg(part + b);  // written by other SMs: read it where they left it, in L2
    m = t > m ? t : m;
  }
  m = block_max(m);
  if (threadIdx.x == 0) {
    *dt_out = __ddiv_rn(cfl, m);
    if (nonphysical_out) *nonphysical_out = (int)(__ldcg(&hdr[1]) & 1u);
    hdr[0] = 0u;  // left clean for the next call (the host clears them again before it launches)
    hdr[1] = 0u;
  }
}

}  // namespace mfc

// Device address of static_scratch on `device`, which must be current: asked of the runtime on the first call for that
// device, remembered afterwards.  The mutex only orders host threads that get here together; it allocates nothing.
constexpr int MFC_STATIC_MAX_DEVICES = 64;
static unsigned char* g_static_dev_ptr[MFC_STATIC_MAX_DEVICES] = {};
static std::mutex g_static_mutex;

static mfc_status static_scratch_on(int device, unsigned char** out) {
  std::lock_guard<std::mutex> lock(g_static_mutex);
  if (!g_static_dev_ptr[device]) {
    void* ptr = nullptr;
    CK(cudaGetSymbolAddress(&ptr, mfc::static_scratch));
    if (!ptr) return fail(MFC_ERR_CUDA, "mfc_cfl_dt_static: cudaGetSymbolAddress returned no address");
    g_static_dev_ptr[device] = static_cast<unsigned char*>(ptr);
  }
  *out = g_static_dev_ptr[device];
  return MFC_OK;
}

template <int N, int D>
static cudaError_t launch_cfl_static(const KP& kp, const double* q, double cfl, unsigned char* scratch, double* dt_out,
                                     int* nonphysical_out, cudaStream_t stream) {
  const unsigned nb = (unsigned)((kp.ncells + ST_CPB - 1) / ST_CPB);
  cfl_static_kernel<N, D><<<nb, PB, 0, stream>>>(kp, q, cfl, scratch, dt_out, nonphysical_out);
  return cudaGetLastError();
}

extern "C" mfc_status mfc_cfl_dt_static(const mfc_params* p, const double* q, double cfl, double* dt_out,
                                        int* nonphysical_out) {
  if (!p || !q || !dt_out) return fail(MFC_ERR_ARG, "mfc_cfl_dt_static: NULL argument");
  if (p->ndim < 1 || p->ndim > 3) return fail(MFC_ERR_ARG, "mfc_cfl_dt_static: ndim must be 1..3");
  if (p->nfluids < 1 || p->nfluids > MFC_MAX_FLUIDS) return fail(MFC_ERR_ARG, "mfc_cfl_dt_static: nfluids must be 1..3");
  if (!p->gamma || !p->pi_inf) return fail(MFC_ERR_ARG, "mfc_cfl_dt_static: gamma/pi_inf NULL");
  long long cells = 1;
  for (int d = 0; d < 3; ++d) {
    if (p->n[d] < 1) return fail(MFC_ERR_ARG, "mfc_cfl_dt_static: n[d] must be >= 1");
    if (d >= p->ndim && p->n[d] != 1) return fail(MFC_ERR_ARG, "mfc_cfl_dt_static: n[d] must be 1 for d >= ndim");
    if (d < p->ndim && !(p->dx[d] > 0.0)) return fail(MFC_ERR_ARG, "mfc_cfl_dt_static: dx[d] must be > 0");
    cells *= p->n[d];
    if (cells > MFC_STATIC_MAX_CELLS)
      return fail(MFC_ERR_ARG,
                  "mfc_cfl_dt_static: grid too large for the built-in scratch array (at most " +
                      std::to_string(MFC_STATIC_MAX_CELLS) + " cells = " + std::to_string(MFC_STATIC_MAX_BLOCKS) +
                      " blocks of " + std::to_string(MFC_STATIC_CELLS_PER_BLOCK) +
                      "); use mfc_init_grid + mfc_cfl_dt, which allocate their own");
  }
  for (int i = 0; i < p->nfluids; ++i)
    if (!(p->gamma[i] > 1.0)) return fail(MFC_ERR_ARG, "mfc_cfl_dt_static: gamma_i must be > 1");
  int ndev = 0;
  CK(cudaGetDeviceCount(&ndev));
  if (p->device < 0 || p->device >= ndev || p->device >= MFC_STATIC_MAX_DEVICES)
    return fail(MFC_ERR_ARG, "mfc_cfl_dt_static: no such CUDA device");
  CK(cudaSetDevice(p->device));
  unsigned char* scratch = nullptr;
  if (mfc_status s = static_scratch_on(p->device, &scratch)) return s;

  KP kp;
  std::memset(&kp, 0, sizeof(KP));
  for (int d = 0; d < 3; ++d) {
    kp.n[d] = p->n[d];
    kp.dx[d] = d < p->ndim ? p->dx[d] : 1.0;
    kp.inv_dx[d] = 1.0 / kp.dx[d];
  }
  kp.ncells = cells;
  for (int i = 0; i < p->nfluids; ++i) {  // as in mfc_init_grid (PAPER.md:117 with eq.(4))
    kp.G[i] = 1.0 / (p->gamma[i] - 1.0);
    kp.P[i] = (p->gamma[i] * p->pi_inf[i]) / (p->gamma[i] - 1.0);
  }
  cudaStream_t stream = (cudaStream_t)p->stream;
  // the array keeps whatever the last call left: the counter and the flag must start at zero even if that call died
  CK(cudaMemsetAsync(scratch, 0, 2 * sizeof(unsigned), stream));
  struct { int nf, ndim; } sel{p->nfluids, p->ndim};
  CK(MFC_DISPATCH(&sel, (launch_cfl_static<N, D>(kp, q, cfl, scratch, dt_out, nonphysical_out, stream))));
  return MFC_OK;
}
