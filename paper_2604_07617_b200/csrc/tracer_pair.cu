// Persistent fp64 DP5 guiding-centre tracer for the Boozer models: WARP PAIRS.  Serves the vacuum model (R1), the
// non-vacuum model with tabulated profiles (R1b) and the shear Alfven wave (R2) of DESIGN.md section 2, each with
// four tabulated quantities or, in the derivative-of-interpolant mode (R1c, template flag DOI), with |B| alone.
//
// What is computed is PAPER.md:57-61 (DESIGN.md sections 1-2); the launch shape is this library's own.
//
// Two blocks of 128 threads per SM, 255 registers per thread.  A block holds two warp pairs; a pair serves 32
// particle slots:
//   * the SCALAR warp: lane l owns particle slot l -- state, DP5 stage states and sums, cell locate (square root,
//     arctangent), the wave terms, the guiding-centre physics, error norm, controller, stop test and refill.
//   * the CONTRACTION warp: lane l owns ALL 256 tricubic coefficients (4 quantities x 64, 2 KiB) of slot l's
//     current cell on chip -- the first PairTraits::NREG in registers, the others in a private conflict-free run of shared
//     memory -- re-fetched from the cell-major table only when the slot's cell changes: the register part by
//     256-bit read-only loads straight into its final registers, the shared part by ONE bulk asynchronous copy
//     (cp.async.bulk) signalled on a thread-private mbarrier.
// Both sides have the registers their instruction-level parallelism needs (a warp with four independent DFMA
// chains saturates its scheduler's FP64 pipe), and each scheduler hosts one warp of either kind, so that the
// latency-bound scalar chains and the throughput-bound contraction fill each other's gaps.
//
// One right-hand-side evaluation ("round") is a two-sided pipeline.  The three local coordinates of a stage point
// do not become known at the same time: the FIRST (zeta) is a state variable, the SECOND (s) needs a square root,
// the LAST (theta) an arctangent.  The scalar warp publishes (wFIRST, wSECOND) as soon as it has them (barrier REQ)
// and goes on with the arctangent, the cell index, the next-cell guess (barrier G), the wave terms and the stage
// sums, while the contraction warp contracts along FIRST and SECOND (60 of the 63 FMA per quantity) on the cell
// it holds and hands back the four plane values of every quantity (barrier DONE); the scalar warp finishes with
// three FMA per quantity in wLAST.  The cell a contraction lane holds at REQ is the scalar warp's guess from the
// round before (fp32 straight-line extrapolation along the attempted step; after the accept / reject decision
// barrier G2), fetched while the scalar warp works; when the located cell differs (rare) the lane redoes the
// contraction with the right cell (barrier D2).  While the scalar warp is on its own (physics, end of an attempt,
// next stage state) the contraction warp waits for the cell that is being fetched and loads the shared-memory rows
// of its first quad: neither depends on the evaluation point, so the request finds it ready.
#include "tracer_common.cuh"

namespace catapult {

struct PairTraits {
  static constexpr int NQ = CATAPULT_NQUANT_BOOZER;
  static constexpr int NCOEF = NQ * 64;
  static constexpr int NREG = 88;                   // coefficients a contraction thread keeps in registers
  static constexpr int NSH = NCOEF - NREG;         // ... and in shared memory
  static constexpr int NT = 128;                   // threads per block: two pairs of warps
  static constexpr int NS = 64;                    // particle slots per block
  // one slot's run of shared memory: NSH doubles + 16 bytes of padding, so that the 8 lanes of a quarter warp
  // reading 16 bytes each at the same offset of their runs hit 8 different 16-byte bank groups (STRIP/16 is odd)
  static constexpr int STRIP = NSH * 8 + 16;
  static_assert(NREG >= 64 && NREG % 4 == 0 && NREG > 0 && NREG < NCOEF, "register part: whole rows");
  static_assert((STRIP / 16) % 2 == 1, "run length must be an odd number of 16-byte groups");
  static constexpr size_t OFF_COEF = 0;                               // [NS] runs of STRIP bytes
  static constexpr size_t OFF_MBAR = OFF_COEF + (size_t)STRIP * NS;   // uint64 [NS]: one mbarrier per slot
  static constexpr size_t OFF_KS = OFF_MBAR + 8 * NS;                 // double [6][4][NS]: stage derivatives k_1..k_6
  static constexpr size_t OFF_PART = OFF_KS + (size_t)6 * 4 * NS * 8;  // double2 [4 planes][2][NS]: plane values
  static constexpr size_t OFF_W = OFF_PART + (size_t)8 * NS * 16;     // double [2][NS]: wFIRST, wSECOND
  static constexpr size_t OFF_G = OFF_W + (size_t)2 * NS * 8;         // int2 [2 parities][NS]: (redo cell, next cell)
  static constexpr size_t OFF_G2 = OFF_G + (size_t)2 * NS * 8;        // int2 [NS]: after accept / reject: (next cell, cell at the end of the next step)
  static constexpr size_t OFF_REQ = OFF_G2 + (size_t)NS * 8;          // int [NS]: request word
  static constexpr size_t SMEM_BYTES = OFF_REQ + (size_t)NS * 4;
  static_assert(2 * (SMEM_BYTES + 1024) <= 233472, "two blocks per SM: 228 KB of shared memory");
};

// named barriers of pair p: ids 1 + 6 p ... (0 is __syncthreads'); every one joins the pair's 64 threads
constexpr int PB_REQ = 0, PB_DONE = 1, PB_G = 2 /* and 3: by round parity */, PB_D2 = 4, PB_G2 = 5;
__device__ __forceinline__ void pbar_sync(int id) { asm volatile("bar.sync %0, 64;" ::"r"(id) : "memory"); }
__device__ __forceinline__ void pbar_arrive(int id) { asm volatile("bar.arrive %0, 64;" ::"r"(id) : "memory"); }

// ---- contraction warp -------------------------------------------------------------------------------------------
// What a contraction thread carries about the cell it holds on chip.
struct PairCell {
  unsigned strip_s, mbar;  // the slot's run of shared memory and its mbarrier (shared-window addresses)
  int cached;              // the cell held (or being fetched); -1: none
  unsigned phase;          // parity of the mbarrier phase the next wait is for
  bool pending;            // a bulk copy into the run is in flight
};

__device__ __forceinline__ void pair_wait(PairCell& pc) {
  if (pc.pending) {
    mbar_wait(pc.mbar, pc.phase);
    pc.phase ^= 1u;
    pc.pending = false;
  }
}

// Fetch of cell c: the first NREG coefficients land in their final registers (256-bit loads), the others go
// global -> shared as ONE bulk asynchronous copy.  Nothing waits here, except for an earlier copy that is still
// landing in the same run.
template <bool DOI>
__device__ __forceinline__ void pair_fetch(const double* __restrict__ table, PairCell& pc,
                                           double (&creg)[PairTraits::NREG], int c) {
  using PT = PairTraits;
  if (DOI) {  // one quantity: 512 bytes, all of it into registers
    const double* src1 = table + (long long)c * 64;
#pragma unroll
    for (int e = 0; e < 64; e += 4) ldg_f64x4(src1 + e, creg[e], creg[e + 1], creg[e + 2], creg[e + 3]);
    pc.cached = c;
    return;
  }
  const double* src = table + (long long)c * PT::NCOEF;
#pragma unroll
  for (int e = 0; e < PT::NREG; e += 4) ldg_f64x4(src + e, creg[e], creg[e + 1], creg[e + 2], creg[e + 3]);
  pair_wait(pc);
  mbar_expect_tx(pc.mbar, PT::NSH * 8);
  bulk_g2s(pc.strip_s, src + PT::NREG, PT::NSH * 8, pc.mbar);
  pc.pending = true;
  pc.cached = c;
}

// Four rows (one of each quantity, same powers of wL and wS) by Horner in wF, interleaved so that four
// independent chains are in flight, then one Horner step in wS of the four planes they belong to.  Written as ONE
// statement in the order the FP64 pipe should see, because neither the compiler's front end (which would gather
// all loads of the evaluation ahead of the arithmetic, a register per loaded value) nor the assembler (which keeps
// close to the order it is given) interleaves dependent chains by itself.  FIRST: the rows open their planes.
template <bool FIRST>
__device__ __forceinline__ void quad_rows(const double (&c)[4][4], double wF, double wS, double (&P)[4]) {
  if (FIRST) {
    asm volatile(
        "{\n\t.reg .f64 t0, t1, t2, t3;\n\t"
        "fma.rn.f64 t0, %7, %20, %6;\n\tfma.rn.f64 t1, %11, %20, %10;\n\t"
        "fma.rn.f64 t2, %15, %20, %14;\n\tfma.rn.f64 t3, %19, %20, %18;\n\t"
        "fma.rn.f64 t0, t0, %20, %5;\n\tfma.rn.f64 t1, t1, %20, %9;\n\t"
        "fma.rn.f64 t2, t2, %20, %13;\n\tfma.rn.f64 t3, t3, %20, %17;\n\t"
        "fma.rn.f64 %0, t0, %20, %4;\n\tfma.rn.f64 %1, t1, %20, %8;\n\t"
        "fma.rn.f64 %2, t2, %20, %12;\n\tfma.rn.f64 %3, t3, %20, %16;\n\t}"
        : "=d"(P[0]), "=d"(P[1]), "=d"(P[2]), "=d"(P[3])
        : "d"(c[0][0]), "d"(c[0][1]), "d"(c[0][2]), "d"(c[0][3]), "d"(c[1][0]), "d"(c[1][1]), "d"(c[1][2]),
          "d"(c[1][3]), "d"(c[2][0]), "d"(c[2][1]), "d"(c[2][2]), "d"(c[2][3]), "d"(c[3][0]), "d"(c[3][1]),
          "d"(c[3][2]), "d"(c[3][3]), "d"(wF));
  } else {
    asm volatile(
        "{\n\t.reg .f64 t0, t1, t2, t3;\n\t"
        "fma.rn.f64 t0, %7, %20, %6;\n\tfma.rn.f64 t1, %11, %20, %10;\n\t"
        "fma.rn.f64 t2, %15, %20, %14;\n\tfma.rn.f64 t3, %19, %20, %18;\n\t"
        "fma.rn.f64 t0, t0, %20, %5;\n\tfma.rn.f64 t1, t1, %20, %9;\n\t"
        "fma.rn.f64 t2, t2, %20, %13;\n\tfma.rn.f64 t3, t3, %20, %17;\n\t"
        "fma.rn.f64 t0, t0, %20, %4;\n\tfma.rn.f64 t1, t1, %20, %8;\n\t"
        "fma.rn.f64 t2, t2, %20, %12;\n\tfma.rn.f64 t3, t3, %20, %16;\n\t"
        "fma.rn.f64 %0, %0, %21, t0;\n\tfma.rn.f64 %1, %1, %21, t1;\n\t"
        "fma.rn.f64 %2, %2, %21, t2;\n\tfma.rn.f64 %3, %3, %21, t3;\n\t}"
        : "+d"(P[0]), "+d"(P[1]), "+d"(P[2]), "+d"(P[3])
        : "d"(c[0][0]), "d"(c[0][1]), "d"(c[0][2]), "d"(c[0][3]), "d"(c[1][0]), "d"(c[1][1]), "d"(c[1][2]),
          "d"(c[1][3]), "d"(c[2][0]), "d"(c[2][1]), "d"(c[2][2]), "d"(c[2][3]), "d"(c[3][0]), "d"(c[3][1]),
          "d"(c[3][2]), "d"(c[3][3]), "d"(wF), "d"(wS));
  }
}

// Makes the calling thread wait HERE for the 256-bit loads that fill its coefficient registers, instead of at their
// first use inside the contraction (which sits behind the REQ barrier, on the critical path of the round).  `last` is
// the register the LAST issued load writes; loads of one thread to distinct registers return in order on this part,
// so when it has landed all have.  The compiler cannot be told "wait for the scoreboard" directly: the only way is an
// instruction that consumes the register, and it must not be removable.  Comparing the high word with a constant and
// branching to a side effect does that.  The constant is the high word of a quiet NaN with an arbitrary payload; a
// table never holds it unless the caller's nodes were NaN, and if one ever did, the only consequence is a sleep of
// about a nanosecond: the test can cost time, it cannot change a result.
__device__ __forceinline__ void wait_for_register_loads(double last) {
  if (__double2hiint(last) == 0x7ffdead0) asm volatile("nanosleep.u32 1;");
}

// Plane values P[a][q] = sum_bc C[q][a][b][c] wS^b wF^c of the four quantities on the cell held: every row (c) by
// Horner in wF, the four rows of a plane by Horner in wS from b = 3 down -- the operations and the order of
// horner_plane (gc_device.cuh), which every user of the table follows.  The 64 rows are walked with the quantity
// running fastest (quad_rows: 16 quads, plane a = 3 first); the rows of a quad that live in shared memory are
// loaded PairRows::AHEAD quads ahead into rotating row buffers; a finished plane goes to the exchange buffer at once.
struct PairRows {  // rotating row buffers of the contraction: [quad modulo (AHEAD + 1)][quantity][4 coefficients]
  static constexpr int AHEAD = 1;  // quads the shared-memory rows are loaded ahead of their use
  double rb[AHEAD + 1][4][4];
  static __device__ __forceinline__ constexpr int first_coef(int s, int q) {  // quad s = (a, b) descending
    return q * 64 + ((3 - s / 4) * 4 + (3 - s % 4)) * 4;
  }
  __device__ __forceinline__ void load_quad(unsigned strip_s, int s) {
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int g = first_coef(s, q);
      if (g >= PairTraits::NREG) lds_row(strip_s + (unsigned)(g - PairTraits::NREG) * 8u, rb[s % (AHEAD + 1)][q]);
    }
  }
  // the rows the first quads need do not depend on the evaluation point: they can be loaded before it is known
  __device__ __forceinline__ void preload(unsigned strip_s) {
#pragma unroll
    for (int s = 0; s < AHEAD; ++s) load_quad(strip_s, s);
  }
};

__device__ __forceinline__ void pair_contract(const double (&creg)[PairTraits::NREG], PairRows& rows,
                                              unsigned strip_s, unsigned part_s, double wS, double wF) {
  using PT = PairTraits;
  constexpr int AHEAD = PairRows::AHEAD;
  double P[4];
#pragma unroll
  for (int s = 0; s < 16; ++s) {
    if (s + AHEAD < 16) rows.load_quad(strip_s, s + AHEAD);
    double c[4][4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int g = PairRows::first_coef(s, q);
#pragma unroll
      for (int e = 0; e < 4; ++e) c[q][e] = (g < PT::NREG) ? creg[g < PT::NREG ? g + e : 0] : rows.rb[s % (AHEAD + 1)][q][e];
    }
    if (s % 4 == 0) quad_rows<true>(c, wF, wS, P);
    else quad_rows<false>(c, wF, wS, P);
    if (s % 4 == 3) {  // plane a = 3 - s/4 of the four quantities: double2 part[a][2][NS]
      const int a = 3 - s / 4;
      sts_f64x2(part_s + (unsigned)((a * 2 + 0) * PT::NS) * 16u, P[0], P[1]);
      sts_f64x2(part_s + (unsigned)((a * 2 + 1) * PT::NS) * 16u, P[2], P[3]);
    }
  }
}

// Derivative-of-interpolant mode (R1c): ONE tabulated quantity, |B|, whose 64 coefficients all sit in the
// thread's registers; the contraction delivers, per power a of wLAST, the plane value, its derivative with respect to
// wSECOND and the plane value of the rows' derivatives with respect to wFIRST (simultaneous value / derivative Horner:
// p <- c3, d <- c3; then d <- d w + p after every p <- p w + c).  112 FMA, no shared-memory traffic.
__device__ __forceinline__ void pair_contract_doi(const double (&creg)[PairTraits::NREG], unsigned part_s, double wS,
                                                  double wF) {
  using PT = PairTraits;
#pragma unroll
  for (int a = 0; a < 4; ++a) {
    double V = 0.0, VS = 0.0, VF = 0.0;
#pragma unroll
    for (int b = 3; b >= 0; --b) {
      const int g = (a * 4 + b) * 4;
      double r = creg[g + 3], dr = creg[g + 3];
      r = fma(r, wF, creg[g + 2]);
      dr = fma(dr, wF, r);
      r = fma(r, wF, creg[g + 1]);
      dr = fma(dr, wF, r);
      r = fma(r, wF, creg[g]);
      if (b == 3) {
        V = r;
        VS = r;
        VF = dr;
      } else {
        V = fma(V, wS, r);
        if (b > 0) VS = fma(VS, wS, V);
        VF = fma(VF, wS, dr);
      }
    }
    sts_f64x2(part_s + (unsigned)((a * 2 + 0) * PT::NS) * 16u, V, VS);
    sts_f64x2(part_s + (unsigned)((a * 2 + 1) * PT::NS) * 16u, VF, 0.0);
  }
}

template <bool DOI>
__device__ __forceinline__ void contraction_warp(const TraceConst& tc, unsigned char* smem, int slot, int bar0) {
  using PT = PairTraits;
  const unsigned FULL = 0xffffffffu;
  const double* __restrict__ table = tc.f.table;
  double creg[PT::NREG];
#pragma unroll
  for (int e = 0; e < PT::NREG; ++e) creg[e] = 0.0;
  PairCell pc;
  pc.strip_s = smem_u32(smem + PT::OFF_COEF + (size_t)slot * PT::STRIP);
  pc.mbar = smem_u32(smem + PT::OFF_MBAR) + 8u * slot;
  pc.cached = -1;
  pc.phase = 0;
  pc.pending = false;
  mbar_init(pc.mbar, 1);
  for (int e = 0; e < PT::NSH; ++e) reinterpret_cast<double*>(smem + PT::OFF_COEF + (size_t)slot * PT::STRIP)[e] = 0.0;
  const unsigned part_s = smem_u32(smem + PT::OFF_PART) + 16u * slot;
  const double* wbuf = reinterpret_cast<const double*>(smem + PT::OFF_W) + slot;
  const volatile int* reqbuf = reinterpret_cast<const volatile int*>(smem + PT::OFF_REQ) + slot;
  const volatile long long* gbuf = reinterpret_cast<const volatile long long*>(smem + PT::OFF_G) + slot;
  const volatile long long* g2buf = reinterpret_cast<const volatile long long*>(smem + PT::OFF_G2) + slot;

  PairRows rows;
  for (;;) {
    // ---- while the scalar warp is on its own: wait for the cell that is being fetched and load the rows the
    // first quads need (neither depends on the evaluation point), so that the request finds the thread ready
    pair_wait(pc);
    wait_for_register_loads(creg[DOI ? 63 : PT::NREG - 1]);
    if (!DOI) rows.preload(pc.strip_s);
    pbar_sync(bar0 + PB_REQ);
    const int rq = reqbuf[0];
    if (rq & REQ_QUIT) {  // pair-uniform
      pair_wait(pc);      // nothing may still be landing in shared memory when the block retires
      break;
    }
    const bool active = rq & 1;
    const int kind = (rq >> 1) & 7;  // pair-uniform
    const int rpar = (rq >> 6) & 1;
    const double wF = wbuf[0], wS = wbuf[PT::NS];
    if (active) {
      if (DOI) pair_contract_doi(creg, part_s, wS, wF);
      else pair_contract(creg, rows, pc.strip_s, part_s, wS, wF);
    }
    __syncwarp();
    pbar_arrive(bar0 + PB_DONE);
    // ---- the scalar warp has located the point: a wrong cell is redone; then the guessed cell of the next
    // point is fetched while the scalar warp works on
    pbar_sync(bar0 + PB_G + rpar);
    const long long g = gbuf[rpar * PT::NS];
    const int redo_cell = (int)g, next_cell = (int)(g >> 32);
    const bool redo = active && redo_cell >= 0;
    if (__any_sync(FULL, redo)) {  // the scalar warp takes the same decision
      if (redo) {
        pair_fetch<DOI>(table, pc, creg, redo_cell);
        if (DOI) {
          pair_contract_doi(creg, part_s, wS, wF);
        } else {
          pair_wait(pc);
          rows.preload(pc.strip_s);
          pair_contract(creg, rows, pc.strip_s, part_s, wS, wF);
        }
      }
      __syncwarp();
      pbar_arrive(bar0 + PB_D2);
    }
    if (active && next_cell >= 0 && next_cell != pc.cached) pair_fetch<DOI>(table, pc, creg, next_cell);
    if (kind == 5) {  // end of an attempt: the first point of the next one depends on the accept / reject decision
      pbar_sync(bar0 + PB_G2);
      const long long g2 = g2buf[0];
      const int t2 = (int)g2, far = (int)(g2 >> 32);
      if (active && t2 >= 0 && t2 != pc.cached) pair_fetch<DOI>(table, pc, creg, t2);
      // the cell in which the next attempt is expected to end: towards L2 now (30 % of the fetches come from
      // HBM otherwise, and a warp waits for its slowest lane)
      if (active && far >= 0 && far != pc.cached) {
        constexpr int CELL_DOUBLES = DOI ? 64 : PT::NCOEF;
        const char* line = reinterpret_cast<const char*>(table + (long long)far * CELL_DOUBLES);
#pragma unroll
        for (int l = 0; l < CELL_DOUBLES * 8 / 128; ++l) asm volatile("prefetch.global.L2 [%0];" ::"l"(line + 128 * l));
      }
    }
  }
}

// ---- scalar warp ------------------------------------------------------------------------------------------------
// What an evaluation accumulates on the side, as zero-padded rows of six coefficients of k_1..k_6: during stage
// point r (0..4) the known part of the next stage state (row r + 1 of the tableau without its last entry), during
// the last one (5) the error sums of Eq. 4 over the first six derivatives, during a start point (6)
// nothing.  A zero coefficient meets a derivative of an earlier attempt: those are kept finite (see the kernel).
static __constant__ double PAIR_SUMS[7][6] = {
    {3.0 / 40.0, 0, 0, 0, 0, 0},
    {44.0 / 45.0, -56.0 / 15.0, 0, 0, 0, 0},
    {19372.0 / 6561.0, -25360.0 / 2187.0, 64448.0 / 6561.0, 0, 0, 0},
    {9017.0 / 3168.0, -355.0 / 33.0, 46732.0 / 5247.0, 49.0 / 176.0, 0, 0},
    {35.0 / 384.0, 0.0, 500.0 / 1113.0, 125.0 / 192.0, -2187.0 / 6784.0, 0},
    {71.0 / 57600.0, 0.0, -71.0 / 16695.0, 71.0 / 1920.0, -17253.0 / 339200.0, 22.0 / 525.0},
    {0, 0, 0, 0, 0, 0}};

constexpr int REPORT_NO_STATUS = 4;

struct ScalarSide {  // what the scalar warp carries from round to round besides the particle state
  int rpar;          // parity of the round (the guess buffer and its barrier are double-buffered by it)
  int held;          // the cell this slot's contraction lane holds (or is fetching)
  unsigned n_load;   // cells fetched for this slot ...
  unsigned n_block;  // ... of which after the point had been located (the guess missed)
};

// One lock-step right-hand-side evaluation of the scalar warp at the point (tr, X): see the top of this file.
// Lanes with act = false publish a request nobody serves.  ratio >= 0: the next point is expected at
// X + ratio (X - base) and its cell is fetched ahead.  S_c = sum_{j < 6} coef[j] k_j,c is accumulated on the side
// (rows of PAIR_SUMS).  All 32 lanes must call this.
template <int MODEL, bool DOI>
__device__ __forceinline__ void scalar_round(const TraceConst& tc, unsigned char* smem, int slot, int bar0, bool act,
                                             int kind, ScalarSide& sr, double tr, const double X[4], double mu,
                                             float ratio, const float base[3], float pos[3], double dy[4],
                                             double& modB, double& level, const double* coef, const double* ks,
                                             double S[4]) {
  using PT = PairTraits;
  using AX = AxisRoles<true>;
  const unsigned FULL = 0xffffffffu;
  const FieldConst& f = tc.f;
  double* wbuf = reinterpret_cast<double*>(smem + PT::OFF_W) + slot;
  int* reqbuf = reinterpret_cast<int*>(smem + PT::OFF_REQ) + slot;
  int2* gbuf = reinterpret_cast<int2*>(smem + PT::OFF_G) + slot;
  EvalGeo g;
  int ci[3];
  double wF, wS, wL;
  // ---- the two coordinates that are known early
  const double r2 = fma(X[0], X[0], X[1] * X[1]);
  fm::sqrt_rsqrt(r2, g.a, g.inva);
  {
    double xr = X[2] - f.lo[AX::FIRST];
    xr = wrap_periodic(xr, f.span[AX::FIRST], f.invspan[AX::FIRST]);
    ci[AX::FIRST] = cell_and_w(xr, f.invh[AX::FIRST], f.k[AX::FIRST], wF, pos[AX::FIRST]);
  }
  ci[AX::SECOND] = cell_and_w(g.a - f.lo[AX::SECOND], f.invh[AX::SECOND], f.k[AX::SECOND], wS, pos[AX::SECOND]);
  wbuf[0] = wF;
  wbuf[PT::NS] = wS;
  sr.rpar ^= 1;
  reqbuf[0] = (act ? 1 : 0) | (kind << 1) | (sr.rpar << 6);
  __syncwarp();
  pbar_arrive(bar0 + PB_REQ);
  // ---- the last coordinate, the cell, the guess
  {
    const double ang = fm::atan2(X[1], X[0]);
    const double xr = wrap_periodic(ang - f.lo[AX::LAST], f.span[AX::LAST], f.invspan[AX::LAST]);
    ci[AX::LAST] = cell_and_w(xr, f.invh[AX::LAST], f.k[AX::LAST], wL, pos[AX::LAST]);
  }
  const int cell = flat_cell(f, ci[0], ci[1], ci[2]);
  const bool bad = act && cell != sr.held;  // the contraction runs on another cell's coefficients: redo
  int target = -1;
  if (act && ratio >= 0.f) target = guess_cell<MODEL>(f, pos, base, ratio);
  gbuf[sr.rpar * PT::NS] = make_int2(bad ? cell : -1, target);
  if (act) {
    const int now = bad ? cell : sr.held;
    const int next = target >= 0 ? target : now;
    sr.n_block += bad;
    sr.n_load += (unsigned)bad + (unsigned)(next != now);
    sr.held = next;
  }
  __syncwarp();
  pbar_arrive(bar0 + PB_G + sr.rpar);
  // ---- in the shadow of the contraction: unit vector, wave terms, stage sums
  g.ca = !(g.a > 0.0) ? 1.0 : X[0] * g.inva;
  g.sa = X[1] * g.inva;
  if (MODEL == MODEL_BOOZER_NV) eval_profiles(f, g);
  if (MODEL == MODEL_BOOZER_SAW) {
    const double ds = g.a - tc.saw_s0;
    g.Phihat = tc.saw_Phi0 * fm::exp(-ds * ds * tc.saw_invw2);
    g.dPhihat = g.Phihat * (-2.0 * ds * tc.saw_invw2);
    // sin / cos of m theta - n zeta + omega t by the addition theorem: cos / sin of theta are y0/s, y1/s
    const double beta = fma(-(double)tc.saw_n, X[2], tc.saw_omega * tr);
    double sb, cb, cm, sm;
    fm::sincos(beta, sb, cb);
    unit_power(tc.saw_m, g.ca, g.sa, cm, sm);
    g.sn = fma(sm, cb, cm * sb);
    g.cs = fma(cm, cb, -sm * sb);
    eval_wave_terms(tc, g);
  }
#pragma unroll
  for (int c = 0; c < 4; ++c) S[c] = 0.0;
#pragma unroll
  for (int j = 0; j < 6; ++j) {  // coef is a zero-padded row of six: no branch on the number of terms
    const double cj = coef[j];
#pragma unroll
    for (int c = 0; c < 4; ++c) S[c] = fma(cj, ks[(size_t)(j * 4 + c) * PT::NS], S[c]);
  }
  const bool anybad = __any_sync(FULL, bad);
  pbar_sync(bar0 + PB_DONE);
  if (anybad) pbar_sync(bar0 + PB_D2);
  // ---- plane values -> field values (the last three FMA of horner64), then the right-hand side
  const double2* part = reinterpret_cast<const double2*>(smem + PT::OFF_PART) + slot;  // [a][2][NS]
  double fv[PT::NQ];
  {
    double2 p[4][2];
#pragma unroll
    for (int a = 0; a < 4; ++a) {
      p[a][0] = part[(a * 2 + 0) * PT::NS];
      p[a][1] = part[(a * 2 + 1) * PT::NS];
    }
    if (DOI) {
      // reading R1c: |B| and its gradient from ONE interpolant; d/dx = (d/dw) 2 / h (w = 2 u - 1)
      fv[0] = horner_row(p[0][0].x, p[1][0].x, p[2][0].x, p[3][0].x, wL);
      const double dL = fma(fma(3.0 * p[3][0].x, wL, 2.0 * p[2][0].x), wL, p[1][0].x);
      const double dS = horner_row(p[0][0].y, p[1][0].y, p[2][0].y, p[3][0].y, wL);
      const double dF = horner_row(p[0][1].x, p[1][1].x, p[2][1].x, p[3][1].x, wL);
      fv[1] = dS * (2.0 * f.invh[AX::SECOND]);
      fv[2] = dL * (2.0 * f.invh[AX::LAST]);
      fv[3] = dF * (2.0 * f.invh[AX::FIRST]);
    } else {
      fv[0] = horner_row(p[0][0].x, p[1][0].x, p[2][0].x, p[3][0].x, wL);
      fv[1] = horner_row(p[0][0].y, p[1][0].y, p[2][0].y, p[3][0].y, wL);
      fv[2] = horner_row(p[0][1].x, p[1][1].x, p[2][1].x, p[3][1].x, wL);
      fv[3] = horner_row(p[0][1].y, p[1][1].y, p[2][1].y, p[3][1].y, wL);
    }
  }
  eval_physics<MODEL>(tc, X, mu, g, fv, dy, modB, level);
}

template <int MODEL, int MODE, bool DOI>
__global__ void __launch_bounds__(PairTraits::NT, 2)
trace_pair_kernel(const __grid_constant__ TraceConst tc, const __grid_constant__ TraceArgs a, const int lane_cap) {
  using PT = PairTraits;
  constexpr int NS = PT::NS;
  extern __shared__ __align__(16) unsigned char smem[];
  const int lane = threadIdx.x & 31;
  const int warp = threadIdx.x >> 5;
  // A block's warps w and w ^ 2 form pair w & 1.  Which of the two is the scalar warp alternates between the two
  // blocks resident on an SM (counted per SM as they start), so that each of the SM's four schedulers hosts one
  // scalar and one contraction warp and the contraction's DFMA load is spread over all four FP64 pipes.
  __shared__ int flip_s;
  if (threadIdx.x == 0) {
    unsigned smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    flip_s = (int)(atomicAdd(reinterpret_cast<unsigned*>(a.queue + 1) + (smid & 1023u), 1u) & 1u);
  }
  __syncthreads();
  const int flip = flip_s;
  const int pair = warp & 1;
  const int slot = pair * 32 + lane;
  const int bar0 = 1 + 6 * pair;
  if ((warp >> 1) != flip) {
    contraction_warp<DOI>(tc, smem, slot, bar0);
    return;
  }
  const unsigned FULL = 0xffffffffu;
  const long long n = a.n;

  // DESIGN.md S3: default step lengths (L = |G| / |B|(node 0), read from the device scalar the field build left)
  double dtmax = tc.dtmax, dt0 = tc.dt0;
  if (!(dtmax > 0.0)) {
    const double Gaxis = (MODEL == MODEL_BOOZER_NV) ? tc.f.prof[0] : tc.f.G;  // non-vacuum: G on the axis
    const double L = __ddiv_rn(fabs(Gaxis), fabs(*tc.f.node0));
    dtmax = __ddiv_rn(__dmul_rn(0.5 * 3.14159265358979323846, L), tc.vtot);
    dt0 = dt0 > 0.0 ? dt0 : __dmul_rn(1e-3, dtmax);
    dt0 = dt0 > dtmax ? dtmax : dt0;
  }
  double* ks = reinterpret_cast<double*>(smem + PT::OFF_KS) + slot;  // k_j component c at ks[(j*4+c)*NS]
#pragma unroll 1
  for (int j = 0; j < 24; ++j) ks[j * NS] = 0.0;
  double ys[4] = {1.0, 0.0, 0.0, 0.0};  // the state at the start of the step
  double dt = 0.0;                      // the controller's step length
  float base[3] = {0.f, 0.f, 0.f};      // start point of the attempt in cell units (next-cell guess)
  double t = 0.0, mu = 0.0;
  long long idx = -1, attempts_left = 0;
  unsigned nacc = 0, nrej = 0, n_eval = 0;  // of the current particle in this call
  int consecutive = 0, step = 0;
  ScalarSide sr{0, -1, 0u, 0u};
  bool active = false;
  int report = -1;  // >= 0: this thread's particle left its slot with this status (REPORT_NO_STATUS: none to count)
  bool exhausted = lane >= lane_cap;  // fewer particles than slots: every warp of the grid takes its share
  unsigned long long rounds = 0;      // warp-uniform

  // statistics of the particles that left their slots: one atomic per warp per counter
  auto flush_reports = [&]() {
    const unsigned reporting = __ballot_sync(FULL, report >= 0);
    if (reporting) {
      if (a.counters) {
        const bool rp = report >= 0;
        unsigned long long v[CATAPULT_NCOUNTERS - 1] = {rp ? nacc : 0u,
                                                        rp ? nrej : 0u,
                                                        report == 0,
                                                        report == 1,
                                                        report == 2,
                                                        report == 3,
                                                        rp ? n_eval : 0u,
                                                        rp ? sr.n_load : 0u,
                                                        rp ? sr.n_block : 0u};
#pragma unroll
        for (int j = 0; j < CATAPULT_NCOUNTERS - 1; ++j) {
          unsigned long long s = v[j];
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(FULL, s, o);
          if (lane == 0 && s) atomicAdd(a.counters + j, s);
        }
      }
      if (report >= 0) {
        sr.n_load = sr.n_block = 0;
        n_eval = 0;
        report = -1;
      }
    }
  };

  for (;;) {
    flush_reports();
    // ---- refill: lanes without a particle pull the next index (one atomic per warp) ------------------
    const bool want = !active && !exhausted;
    const unsigned need = __ballot_sync(FULL, want);
    bool fresh = false;
    double x[4] = {0.0, 0.0, 0.0, 0.0}, y[4] = {1.0, 0.0, 0.0, 0.0};
    if (need) {
      const int leader = __ffs(need) - 1;
      unsigned long long base = 0;
      if (lane == leader) base = atomicAdd(a.queue, (unsigned long long)__popc(need));
      base = __shfl_sync(FULL, base, leader);
      if (want) {
        const long long mine = (long long)base + __popc(need & ((1u << lane) - 1u));
        if (mine >= n) {
          exhausted = true;
        } else {
          idx = mine;
#pragma unroll
          for (int c = 0; c < 4; ++c) x[c] = a.x_in[c * n + idx];
          bool skip = false;
          if (MODE == MODE_STEP_ONCE) {
            t = a.t_io[idx];
          } else if (a.resume) {
            skip = (a.status[idx] != CATAPULT_ST_REACHED_T);
            t = a.t_io[idx];
            if (!(t < tc.T)) skip = true;  // already at (or past) the requested end time
          } else {
            t = 0.0;
          }
          if (!skip) {
            state_to_y<MODEL>(x, y);
            fresh = true;
          }
        }
      }
    }
    if (__any_sync(FULL, fresh)) {
      // the start point's field values give mu and k1
      double dy0[4], B, level, S[4];
      float pos[3];
      scalar_round<MODEL, DOI>(tc, smem, slot, bar0, fresh, KIND_START, sr, t, y, 0.0, -1.f, base, pos, dy0, B, level,
                          PAIR_SUMS[6], ks, S);
      ++rounds;
      if (fresh) {
        n_eval = 1;
        nacc = nrej = 0;
        if (MODE != MODE_STEP_ONCE && a.resume) {
          mu = a.mu_io[idx];
          dt = a.dt_io[idx];
        } else {
          mu = (tc.vtot2 - x[3] * x[3]) / (2.0 * B);
          dt = dt0;
        }
        if (MODE != MODE_STEP_ONCE && !a.resume && is_lost<MODEL>(tc, level)) {
          // born outside: returned unchanged, t_stop = 0
#pragma unroll
          for (int c = 0; c < 4; ++c) a.x_out[c * n + idx] = x[c];
          a.t_io[idx] = 0.0;
          a.status[idx] = CATAPULT_ST_LOST;
          if (a.dt_io) a.dt_io[idx] = dt;
          if (a.mu_io) a.mu_io[idx] = mu;
          if (a.nacc) a.nacc[idx] = 0;
          if (a.nrej) a.nrej[idx] = 0;
          report = CATAPULT_ST_LOST;
        } else if (MODE != MODE_STEP_ONCE && a.init_only) {
          a.t_io[idx] = 0.0;
          a.status[idx] = CATAPULT_ST_REACHED_T;
          a.dt_io[idx] = dt;
          a.mu_io[idx] = mu;
          report = REPORT_NO_STATUS;
        } else {
          active = true;
        }
      }
      // k1 with the particle's own mu (mu enters the right-hand side linearly; the round is simply repeated:
      // once per particle)
      const bool go = fresh && active;
      if (__any_sync(FULL, go)) {
        scalar_round<MODEL, DOI>(tc, smem, slot, bar0, go, KIND_START, sr, t, y, mu, -1.f, base, pos, dy0, B, level,
                            PAIR_SUMS[6], ks, S);
        ++rounds;
        if (go) {
          ++n_eval;
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            ks[c * NS] = dy0[c];
            ys[c] = y[c];
          }
#pragma unroll
          for (int d = 0; d < 3; ++d) base[d] = pos[d];  // the first attempt is extrapolated from here
          consecutive = 0;
          step = 0;
          attempts_left = tc.max_steps > 0 ? tc.max_steps : -1;
        }
      }
    }
    if (!__any_sync(FULL, active)) {
      if (__all_sync(FULL, exhausted)) break;
      continue;
    }

    // ---- one attempted step for every active lane -------------------------------------------------------
    int finish = -1;
    double h = 0.0;
    bool clamped = false;
    if (active) {
      if (MODE == MODE_SCRIPT) {
        h = (step < a.script_len) ? a.script_h[(long long)step * n + idx] : 0.0;
        if (!(h > 0.0)) finish = CATAPULT_ST_REACHED_T;
      } else if (MODE == MODE_STEP_ONCE) {
        h = a.script_h[idx];
      } else if (attempts_left == 0) {
        finish = CATAPULT_ST_MAXSTEPS;
      } else {
        const double rem = tc.T - t;
        clamped = !(dt < rem);  // the last step lands exactly on T (S4)
        h = clamped ? rem : dt;
      }
    }
    const bool stepping = active && finish < 0;
    if (__any_sync(FULL, stepping)) {
      double X[4], dy[4], S[4] = {0.0, 0.0, 0.0, 0.0}, B_, level = 0.0;
      float pos[3];
#pragma unroll
      for (int c = 0; c < 4; ++c) dy[c] = ks[c * NS];  // k1 (first-same-as-last, or the start point's derivative)
#pragma unroll 1
      for (int r = 0; r < 6; ++r) {
        // stage state y + h sum_{j<=r} a[r][j] k_j (row 5 = b: the new state); the sum over j < r was
        // accumulated during the previous evaluation (S), the newest derivative enters last
        const double ad = DP_A[r][r];
#pragma unroll
        for (int c = 0; c < 4; ++c) X[c] = fma(h, fma(ad, dy[c], S[c]), ys[c]);
        const float ratio = (MODE == MODE_STEP_ONCE && r == 5) ? -1.f : NEXT_POINT_RATIO[r];
        // on the side: the known part of the next stage state; in the last round the error sums of Eq. 4
        // over the first six derivatives
        scalar_round<MODEL, DOI>(tc, smem, slot, bar0, stepping, r, sr, fma(DP_C[r], h, t), X, mu, ratio, base, pos, dy, B_,
                            level, PAIR_SUMS[r], ks, S);
        if (r < 5) {  // k_7 stays in registers: it is the next step's k_1 (or nothing)
#pragma unroll
          for (int c = 0; c < 4; ++c) ks[((r + 1) * 4 + c) * NS] = dy[c];
        }
      }
      rounds += 6;
      // PAPER.md:85 Eq. 4 with c = (1,1,1,v_total), state and derivative at the start of the step
      double r = 0.0, chk = 0.0;
      {
        const double ah = fabs(h);
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const double sc = (c == 3) ? tc.atol * tc.vtot : tc.atol;
          const double rden = fm::rcp(fma(tc.rtol, fma(ah, fabs(ks[c * NS]), fabs(ys[c])), sc));
          const double e = fma(DP_E[6], dy[c], S[c]) * h;
          const double v = fabs(e) * rden;
          chk += v;
          r = fmax(r, v);
        }
      }
      r = (chk == chk) ? r : chk;  // a non-finite component is a rejection
      if (MODE != MODE_STEP_ONCE && (!(chk == chk) || fabs(chk) > 1.7e308)) {
        // the derivatives of this attempt will meet zero coefficients in the next one's sums: keep them finite
#pragma unroll 1
        for (int j = 4; j < 24; ++j) ks[j * NS] = 0.0;
      }
      bool accepted = false;
      double dtn = h;
      if (MODE == MODE_SCRIPT) accepted = true;
      else if (MODE == MODE_ADAPTIVE) dtn = controller(h, r, dtmax, accepted);
      {
        // the decision goes to the contraction warp at once: the cell of the next attempt's first point, a fifth
        // of the next step length beyond the new start point (accepted: the end point; rejected: the old start
        // point)
        int target = -1, far = -1;
        if (MODE != MODE_STEP_ONCE && stepping) {
          double hn = h;
          if (MODE == MODE_ADAPTIVE) {
            const double tn = accepted ? (clamped ? tc.T : t + h) : t;
            hn = fmin((accepted && clamped) ? dt : dtn, tc.T - tn);
          }
          const float fr = 0.2f * __fdividef((float)hn, (float)h);
          target = guess_cell<MODEL>(tc.f, pos, base, accepted ? fr : fr - 1.0f);
          far = guess_cell<MODEL>(tc.f, pos, base, accepted ? 5.0f * fr : 5.0f * fr - 1.0f);
          sr.n_load += (unsigned)(target != sr.held);
          sr.held = target;
          if (accepted) {
#pragma unroll
            for (int d = 0; d < 3; ++d) base[d] = pos[d];
          }
        }
        reinterpret_cast<int2*>(smem + PT::OFF_G2)[slot] = make_int2(target, far);
        __syncwarp();
        pbar_arrive(bar0 + PB_G2);
      }
      if (stepping) {
        n_eval += 6;
        if (attempts_left > 0) --attempts_left;
        if (MODE == MODE_SCRIPT) {
          if (a.script_r) a.script_r[(long long)step * n + idx] = r;
          ++step;
        } else if (MODE == MODE_STEP_ONCE) {
          double xn[4];
          y_to_state<MODEL>(X, xn);
#pragma unroll
          for (int c = 0; c < 4; ++c) a.x_out[c * n + idx] = xn[c];
          a.script_r[idx] = r;
#pragma unroll
          for (int j = 0; j < 7; ++j)
#pragma unroll
            for (int c = 0; c < 4; ++c) a.kall[((long long)j * 4 + c) * n + idx] = j < 6 ? ks[(j * 4 + c) * NS] : dy[c];
          active = false;
          report = REPORT_NO_STATUS;
          if (!(chk == chk) || fabs(chk) > 1.7e308) {
            // same guard as above, after the derivatives have been reported: the next particle in this slot must
            // not meet 0 * NaN in its stage sums
#pragma unroll 1
            for (int j = 4; j < 24; ++j) ks[j * NS] = 0.0;
          }
        }
        if (MODE != MODE_STEP_ONCE) {
          if (!accepted) {
            ++nrej;
            dt = dtn;
            if (++consecutive >= tc.max_rej) finish = CATAPULT_ST_STALLED;  // DESIGN.md S6
          } else {
            consecutive = 0;
            ++nacc;
            const bool lost = is_lost<MODEL>(tc, level);
            if (lost && tc.loss_time_mode == 1) {
              // DESIGN.md S5b: the loss time and state inside this step (Hermite interpolant, bisection)
              const double ka[4] = {ks[0], ks[NS], ks[2 * NS], ks[3 * NS]};
              const double theta = loss_refine_boozer(ys, ka, X, dy, h);  // X <- y(theta)
              t = __dadd_rn(t, __dmul_rn(theta, h));
            } else {
              t = clamped ? tc.T : t + h;
            }
            if (!clamped) dt = dtn;
#pragma unroll
            for (int c = 0; c < 4; ++c) {
              ys[c] = X[c];
              ks[c * NS] = dy[c];  // first-same-as-last
            }
            // DESIGN.md S5: loss first, then T
            if (lost) finish = CATAPULT_ST_LOST;
            else if (MODE != MODE_SCRIPT && t >= tc.T) finish = CATAPULT_ST_REACHED_T;
          }
        }
      }
    }
    if (active && finish >= 0) {
      double xo[4];
      y_to_state<MODEL>(ys, xo);
#pragma unroll
      for (int c = 0; c < 4; ++c) a.x_out[c * n + idx] = xo[c];
      a.t_io[idx] = t;
      a.status[idx] = finish;
      if (a.dt_io) a.dt_io[idx] = dt;
      if (a.mu_io) a.mu_io[idx] = mu;
      if (a.nacc) a.nacc[idx] = (a.resume ? a.nacc[idx] : 0u) + nacc;
      if (a.nrej) a.nrej[idx] = (a.resume ? a.nrej[idx] : 0u) + nrej;
      report = finish;
      active = false;
    }
  }
  flush_reports();
  // release the contraction warp
  reinterpret_cast<int*>(smem + PT::OFF_REQ)[slot] = REQ_QUIT;
  __syncwarp();
  pbar_arrive(bar0 + PB_REQ);

  if (a.counters && lane == 0 && rounds) atomicAdd(a.counters + CATAPULT_NCOUNTERS - 1, rounds);
}


// ---- launchers ---------------------------------------------------------------------------------------------
// Persistent grid: two blocks per SM (or fewer when there are fewer particles than warps could share out).
template <int MODEL, int MODE, bool DOI>
static catapult_status pair_shape(int64_t n, int* blocks, int* threads, int* lane_cap) {
  using PT = PairTraits;
  static thread_local int cached_device = -1, cached_resident = 0;
  int dev = 0;
  CATAPULT_CUDA_TRY(cudaGetDevice(&dev));
  if (cached_device != dev) {
    int sms = 0, per_sm = 0;
    CATAPULT_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    CATAPULT_CUDA_TRY(cudaFuncSetAttribute(trace_pair_kernel<MODEL, MODE, DOI>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           (int)PT::SMEM_BYTES));
    CATAPULT_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, trace_pair_kernel<MODEL, MODE, DOI>, PT::NT,
                                                                    PT::SMEM_BYTES));
    if (per_sm < 1) {
      set_error("the tracer kernel does not fit on this device (registers / shared memory)");
      return CATAPULT_ECUDA;
    }
    cached_device = dev;
    cached_resident = sms * per_sm;  // a multiple of the SM count
  }
  long long want = (n + 31) / 32;  // a block is worth starting for 32 particles
  if (want < 1) want = 1;
  const int b = (int)(want < cached_resident ? want : cached_resident);
  // fewer particles than slots: every scalar warp takes an equal share instead of the first warps taking 32 each
  const long long warps = (long long)b * 2;
  long long cap = (n + warps - 1) / warps;
  *lane_cap = (int)(cap < 1 ? 1 : (cap > 32 ? 32 : cap));
  *blocks = b;
  *threads = PT::NT;
  return CATAPULT_OK;
}

template <int MODEL, int MODE, bool DOI>
static catapult_status pair_launch(const TraceConst& tc, const TraceArgs& a, cudaStream_t s) {
  int blocks = 0, threads = 0, cap = 32;
  catapult_status st = pair_shape<MODEL, MODE, DOI>(a.n, &blocks, &threads, &cap);
  if (st != CATAPULT_OK) return st;
  trace_pair_kernel<MODEL, MODE, DOI><<<blocks, threads, PairTraits::SMEM_BYTES, s>>>(tc, a, cap);
  CATAPULT_CUDA_TRY(cudaGetLastError());
  return CATAPULT_OK;
}

template <int MODE>
static catapult_status pair_dispatch(const TraceConst& tc, const TraceArgs& a, int model, cudaStream_t s) {
  if (a.n == 0) return CATAPULT_OK;
  if (tc.f.m == 1) {  // derivative-of-interpolant mode (one tabulated quantity)
    if (model == MODEL_BOOZER_VAC) return pair_launch<MODEL_BOOZER_VAC, MODE, true>(tc, a, s);
    if (model == MODEL_BOOZER_NV) return pair_launch<MODEL_BOOZER_NV, MODE, true>(tc, a, s);
    return pair_launch<MODEL_BOOZER_SAW, MODE, true>(tc, a, s);
  }
  if (model == MODEL_BOOZER_VAC) return pair_launch<MODEL_BOOZER_VAC, MODE, false>(tc, a, s);
  if (model == MODEL_BOOZER_NV) return pair_launch<MODEL_BOOZER_NV, MODE, false>(tc, a, s);
  return pair_launch<MODEL_BOOZER_SAW, MODE, false>(tc, a, s);
}

catapult_status launch_trace_pair(const TraceConst& tc, const TraceArgs& a, int model, int mode, cudaStream_t s) {
  switch (mode) {
    case MODE_ADAPTIVE: return pair_dispatch<MODE_ADAPTIVE>(tc, a, model, s);
    case MODE_SCRIPT: return pair_dispatch<MODE_SCRIPT>(tc, a, model, s);
    default: return pair_dispatch<MODE_STEP_ONCE>(tc, a, model, s);
  }
}

catapult_status trace_pair_shape(int model, bool doi, int64_t n, int* blocks, int* threads) {
  int cap = 0;
  if (doi) {  // the derivative-of-interpolant kernels are other instantiations with their own register count
    if (model == MODEL_BOOZER_VAC) return pair_shape<MODEL_BOOZER_VAC, MODE_ADAPTIVE, true>(n, blocks, threads, &cap);
    if (model == MODEL_BOOZER_NV) return pair_shape<MODEL_BOOZER_NV, MODE_ADAPTIVE, true>(n, blocks, threads, &cap);
    return pair_shape<MODEL_BOOZER_SAW, MODE_ADAPTIVE, true>(n, blocks, threads, &cap);
  }
  if (model == MODEL_BOOZER_VAC) return pair_shape<MODEL_BOOZER_VAC, MODE_ADAPTIVE, false>(n, blocks, threads, &cap);
  if (model == MODEL_BOOZER_NV) return pair_shape<MODEL_BOOZER_NV, MODE_ADAPTIVE, false>(n, blocks, threads, &cap);
  return pair_shape<MODEL_BOOZER_SAW, MODE_ADAPTIVE, false>(n, blocks, threads, &cap);
}

}  // namespace catapult
