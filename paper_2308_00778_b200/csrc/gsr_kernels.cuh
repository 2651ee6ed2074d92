// gsr_kernels.cuh -- sm_100a kernels of the AVU-GSR LSQR hot path (arXiv 2308.00778).
// Citations are lines of PAPER.md; the design is described in DESIGN.md.
// No tensor cores: the path is two sparse products bound by HBM and by gather/scatter rate.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdio>

// -DGSR_BOUNDS_CHECK (paper_2308_00778_b200.build.build(check=True) -> libgsr_check.so): every gather / scatter index
// of the aprod kernels is checked against its section and the kernel traps on a violation.  compute-sanitizer is
// closed on this pool; the parity tests are run against this build instead (profiles/r02_boundscheck.md).
#ifdef GSR_BOUNDS_CHECK
#define GSR_ASSERT(c)                                                                 \
    do {                                                                              \
        if (!(c)) {                                                                   \
            printf("GSR_ASSERT failed: %s (%s:%d)\n", #c, __FILE__, __LINE__);        \
            __trap();                                                                 \
        }                                                                             \
    } while (0)
#else
#define GSR_ASSERT(c) ((void)0)
#endif

namespace gsr {

constexpr int N_ASTRO = 5, N_ATT = 12, N_INSTR = 6, N_PAR = 24;
constexpr int TILE = 32;          // rows per warp tile
constexpr int WARPS = 8;          // warps per CTA of the aprod kernels
constexpr int THREADS = WARPS * 32;
constexpr int ATT_BLOCK_BITS = 21;   // rows per block of the time-ordered attitude copy (2^21)
constexpr int INS_ROW_BITS = 13;     // rows per block of the column-ordered instrument copy (2^13: the block's slice of y is 64 KB of shared memory)
constexpr int INS_BLOCK = 1 << INS_ROW_BITS;
constexpr int INS_KEY_COL = INS_ROW_BITS + 3, INS_KEY_BLOCK = INS_KEY_COL + 16;   // sort key of the build: block | column (16 bits) | row in block | slot (3 bits)
constexpr int INS_BUCKET_MAX = 7680; // instrument columns per bucket: one bucket's accumulators are 60 KB of shared memory

// Device layout of the coefficients ("tile-transposed"): the 32 rows of a warp tile are stored
// coefficient-major, V[(tile*24 + k)*32 + lane], so that lane <-> row reads each of its 24
// coefficients with one coalesced 8-byte load per warp instruction (256 B, two lines) and no
// shared-memory transposition.  instrCol likewise: ic[(tile*6 + j)*32 + lane].  Storage is padded
// to whole tiles (zero coefficients, column 0).  The upload format stays row-major.
// Other section widths (model variants): the same layout with nPar coefficients / nI columns per row.
__host__ __device__ __forceinline__ int64_t vpos(int64_t i, int k, int nPar = N_PAR) { return ((i >> 5) * nPar + k) * TILE + (i & 31); }
__host__ __device__ __forceinline__ int64_t cpos(int64_t i, int j, int nI = N_INSTR) { return ((i >> 5) * nI + j) * TILE + (i & 31); }
constexpr int MAX_GLOB = 16;      // widest global section (GSR_MAX_GLOB in gsr.h)

// Device view of the uploaded system (A_d, M_i, I_c) in upload layout.
struct MatView {
    double *V;             // [nTiles*24*32] tile-transposed, see vpos()
    const int32_t *star;   // [m] star of the row (matrixIndexAstro / 5; -1: the uploaded value broke its contract);
                           // upload scratch only: validated, turned into rp and tw, then freed
    const unsigned long long *tw;   // [nTiles] "tile word" (the star row pointer in place of a per-row
                           // star index, 0.25 B/row): bits 0-31 head mask (bit l: row l of the tile starts a star; bit 0
                           // refers to the last row of the previous tile), bits 32-60 star of the tile's first row,
                           // bit 61: the star of the tile's last row goes on in the next tile, bit 62: some star between
                           // two rows of the tile has no rows (star of a lane then comes from a search in rp)
    const int32_t *iatt;   // [m] attitude start s_i (axis 0; -1: out of range) -- SURVEY 8(f) NEXT-2: 4-byte indices
    const int32_t *ic;     // [nTiles*6*32] tile-transposed, see cpos(); nullptr when ic16 is in use
    const uint16_t *ic16;  // the same as 2-byte columns when nInstr <= 65536 (-12 B/row)
    const int64_t *rp;     // [nStars+1] derived star row pointer
    int64_t m, nStars, nDof, nInstr;
    int64_t offAtt, offInstr, offGlob, n;
    // section widths: 5 / 12 / 6 / 1 in production (the kernels specialised for it use the constants above);
    // a section of width 0 has no columns.  nPar = nA + nAtt + nI + nG coefficients per stored row.
    int nA, nAtt, nI, nG, nPar;
    // constraint rows (CSR, absolute columns)
    const int64_t *conRp, *conCol;
    double *conVal;
    int64_t nCon;
    // time-ordered attitude copy (built at upload when memory allows; nullptr otherwise):
    // attT[k*m + t] = V[permT[t]*24 + 5 + k], rows t sorted by attitude start sT[t] (stable)
    double *attT;
    const int32_t *sT;
    const uint32_t *permT;
    // replicated accumulators of the instrumental section for aprod2: insRep[r*nInstr + c]
    double *insRep;
    int nRep;
    int nInsSm;            // instrument columns [0, nInsSm) accumulate in shared memory (k_aprod2<.., PRIV>)
    // column-ordered copy of the instrumental section (built at upload when memory allows; nullptr otherwise), for
    // k_ins_scatter: the 6 coefficients of the rows of block b (INS_BLOCK consecutive rows) sorted by column, then row;
    // insMeta[e] = column << INS_ROW_BITS | row inside the block; columns are cut into insNB buckets of insW (a multiple of
    // INS_WARPS) and every bucket into INS_WARPS sub-buckets; insPtr[b*insNB*INS_WARPS + j]: first entry of sub-bucket j of
    // block b
    double *insVal;
    const uint32_t *insMeta;
    const int64_t *insPtr;
    int insNB, insW;
};

// Scalars of the LSQR recurrences, resident in device memory.
struct Scalars {
    // coefficients read by the vector / aprod kernels
    double a1_cx, a1_cy;   // aprod1:  u^ <- a1_cx * (A v^) + a1_cy * u^
    double a2_cx, a2_cy;   // aprod2:  v^ <- a2_cx * v^ + a2_cy * (A^T u^)
    double t1, t2, inv_rho, inv_alpha;
    // recurrence state
    double alpha, beta, rhobar, phibar, bnorm, anorm, acond, ddnorm, xxnorm, xnorm, z, cs2, sn2;
    double rnorm, arnorm;
    double atol, btol, ctol;
    long long itn, itnlim;
    int istop;
    int done;              // 1: loop body is a no-op (stopped, or trivial system)
};

constexpr int TW_STAR_BITS = 29;   // n_stars < 2^29
__device__ __forceinline__ int64_t star_search(const int64_t *__restrict__ rp, int64_t nStars, int64_t i)
{
    int64_t lo = 0, hi = nStars;   // largest s with rp[s] <= i among stars that own rows: first s with rp[s+1] > i
    while (lo < hi) {
        const int64_t mid = (lo + hi) >> 1;
        if (rp[mid + 1] <= i) lo = mid + 1; else hi = mid;
    }
    return lo;
}
// star of row (tile, lane) from the tile word
__device__ __forceinline__ int64_t star_of(const MatView &A, unsigned long long w, int64_t i, int lane)
{
    if ((w >> 62) & 1ull) return star_search(A.rp, A.nStars, i);
    return int64_t((w >> 32) & ((1ull << TW_STAR_BITS) - 1)) + __popc(uint32_t(w) & (0xffffffffu >> (31 - lane)) & 0xfffffffeu);
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Totals of up to 5 per-lane values over the 32 lanes of a warp with 9 shuffles instead of 5 x 5 (the values are
// handed round while they are summed: 4 + 2 + 1 exchanges, then two plain butterfly steps).  Afterwards lane 4k holds
// the total of value k; the tree is fixed, so the result is reproducible.
__device__ __forceinline__ double warp_sum5(const double (&s)[5], int lane)
{
    const bool h16 = lane & 16, h8 = lane & 8, h4 = lane & 4;
    double a[4], b[2];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const double lo = s[j], hi = j == 0 ? s[4] : 0.0;   // values 5..7 do not exist
        const double recv = __shfl_xor_sync(0xffffffffu, h16 ? lo : hi, 16);
        a[j] = (h16 ? hi : lo) + recv;
    }
#pragma unroll
    for (int j = 0; j < 2; ++j) {
        const double recv = __shfl_xor_sync(0xffffffffu, h8 ? a[j] : a[2 + j], 8);
        b[j] = (h8 ? a[2 + j] : a[j]) + recv;
    }
    const double recv = __shfl_xor_sync(0xffffffffu, h4 ? b[0] : b[1], 4);
    double c = (h4 ? b[1] : b[0]) + recv;
    c += __shfl_xor_sync(0xffffffffu, c, 2);
    c += __shfl_xor_sync(0xffffffffu, c, 1);
    return c;
}

// Deterministic block sum (fixed tree); result valid in thread 0.  red: >= 32 doubles of smem.
__device__ __forceinline__ double block_sum(double v, double *red)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    v = warp_sum(v);
    __syncthreads();
    if (lane == 0) red[w] = v;
    __syncthreads();
    double r = 0.0;
    if (w == 0) {
        const int nw = (blockDim.x + 31) >> 5;
        r = lane < nw ? red[lane] : 0.0;
        r = warp_sum(r);
    }
    return r;
}

// The 24 coefficients of row (tile, lane): coalesced streaming loads.  ATT: load the attitude
// coefficients too (k = 5..16).
// NA (5 or 0 astrometric coefficients) and NG (1 or 0 global ones) select the layouts that share the specialised kernels:
// 5/12/6/1 (production), 5/12/6/0 and 0/12/6/0 (the section subsets the paper's datasets solve).
// NG = -1: any number of global columns (A.nG, up to MAX_GLOB; "future astrometric models will have more global
// parameters"): their coefficients are not held in v but loaded where they are used, and the row width is
// A.nPar.
template <bool ATT, bool INS = true, int NA = N_ASTRO, int NG = 1>
__device__ __forceinline__ void load_row(const double *__restrict__ g, double (&v)[NA + N_ATT + N_INSTR + (NG > 0 ? NG : 0)])
{
    constexpr int NP = NA + N_ATT + N_INSTR + (NG > 0 ? NG : 0);
#pragma unroll
    for (int q = 0; q < NP; ++q) {
        const bool att = q >= NA && q < NA + N_ATT, ins = q >= NA + N_ATT && q < NA + N_ATT + N_INSTR;
        if ((att && !ATT) || (ins && !INS)) v[q] = 0.0;
        else v[q] = __ldcs(g + q * TILE);
    }
}

// The 6 instrument columns of row (tile, lane): coalesced streaming loads of 2- or 4-byte columns.
template <bool IC16>
__device__ __forceinline__ void load_ic(const MatView &A, int64_t tile, int lane, int32_t (&c)[N_INSTR])
{
    if (IC16) {
        const uint16_t *p = A.ic16 + tile * (N_INSTR * TILE) + lane;
#pragma unroll
        for (int j = 0; j < N_INSTR; ++j) c[j] = int32_t(__ldcs(p + j * TILE));
    } else {
        const int32_t *p = A.ic + tile * (N_INSTR * TILE) + lane;
#pragma unroll
        for (int j = 0; j < N_INSTR; ++j) c[j] = __ldcs(p + j * TILE);
    }
}
// setup kernels: one stored instrument column, either width
__device__ __forceinline__ int32_t ic_at(const MatView &A, int64_t pos) { return A.ic16 ? int32_t(A.ic16[pos]) : A.ic[pos]; }

// ---------------------------------------------------------------------------------------
// aprod mode 1 (Eq. 2; Algorithm 2):  y <- cy*y + cx*(A x), one pass over A,
// all four sections in one kernel, plus the per-CTA partial of sum y^2 (Eq. 4's norm, fused:
// SURVEY a3).  coef = {cx, cy} in device memory.  Row i <-> one lane; a warp owns 32
// consecutive rows, a CTA 256.
// ---------------------------------------------------------------------------------------
// xPack[3*s + a] = x[offAtt + a*nDof + s]: the attitude unknowns of the operand of the fused pass interleaved by
// axis, so that the 12 unknowns of a row (3 axes x 4 consecutive starts; the paper keeps the axes N_DFA
// apart) are one contiguous 96-byte run: 3-4 L2 sectors per row instead of 5-6, and the
// 12 gathers of a lane fall into one or two L1 lines.  24 MB copied per product (~15 us).
__global__ void k_pack_att(MatView A, const double *__restrict__ x, double *__restrict__ xPack, const int *done)
{
    if (done && *done) return;
    const int64_t total = A.nDof * 3;
    for (int64_t e = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; e < total;
         e += int64_t(gridDim.x) * blockDim.x) {
        const int64_t s = e / 3;
        const int a = int(e - s * 3);
        xPack[e] = x[A.offAtt + a * A.nDof + s];
    }
}
// The standalone k_aprod1 is held by the LSU data pipe (86 % of its wavefronts, 12 of them per row for the attitude
// unknowns alone): there the unknowns are packed four wide, xPack4[4*s + a] (a = 3: unused), so that every start is one
// aligned 32-byte sector and a row takes 4 loads of 32 bytes instead of 12 of 8 (Medium: 10.2 -> 9.5 ms).  The fused pass
// keeps the three-wide layout and the texture path: it is held by requests, not by LSU wavefronts, and ran 0.45 ms
// slower with these loads.
__global__ void k_pack_att4(MatView A, const double *__restrict__ x, double *__restrict__ xPack4, const int *done)
{
    if (done && *done) return;
    const int64_t total = A.nDof * 4;
    for (int64_t e = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; e < total;
         e += int64_t(gridDim.x) * blockDim.x) {
        const int64_t s = e >> 2;
        const int a = int(e & 3);
        xPack4[e] = a < 3 ? x[A.offAtt + a * A.nDof + s] : 0.0;
    }
}

template <bool IC16, int NA = N_ASTRO, int NG = 1>
__global__ void __launch_bounds__(THREADS, 2)
k_aprod1(MatView A, const double *__restrict__ x, double *__restrict__ y,
         const double *__restrict__ coef, double *__restrict__ sqPartial, const int *done,
         const double *__restrict__ xPack)
{
    __shared__ double red[32];
    if (done && *done) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const double cx = coef[0], cy = coef[1];
    const int64_t nTiles = (A.m + TILE - 1) / TILE;
    const double *xIns = x + A.offInstr;
    const double xg = NG > 0 ? __ldg(x + A.offGlob) : 0.0;
    constexpr int KT = NA, KI = NA + N_ATT, KG = NA + N_ATT + N_INSTR, NGR = NG > 0 ? NG : 0;
    const int np = NG < 0 ? A.nPar : KG + NG;   // stored coefficients per row
    double sq = 0.0;
    for (int64_t tile = int64_t(blockIdx.x) * WARPS + warp; tile < nTiles;
         tile += int64_t(gridDim.x) * WARPS) {
        const int64_t r0 = tile * TILE;
        const int nrows = int(min(int64_t(TILE), A.m - r0));
        if (lane < nrows) {
            const int64_t i = r0 + lane;
            double v[KG + NGR];
            const double *g = A.V + tile * (int64_t(np) * TILE) + lane;
            load_row<true, true, NA, NG>(g, v);
            const int64_t iatt = __ldcs(A.iatt + i);
            int32_t c[N_INSTR];
            load_ic<IC16>(A, tile, lane, c);
            GSR_ASSERT(iatt >= 0 && iatt + 4 <= A.nDof);
#pragma unroll
            for (int j = 0; j < N_INSTR; ++j) GSR_ASSERT(c[j] >= 0 && c[j] < A.nInstr);
            double sum = 0.0;
            if (NA > 0) {
                const double *xa = x + NA * star_of(A, __ldg(A.tw + tile), i, lane);
                GSR_ASSERT(xa >= x && xa + NA <= x + A.offAtt);
#pragma unroll
                for (int k = 0; k < NA; ++k) sum = fma(v[k], __ldg(xa + k), sum);
            }
            {
                const double *xp = xPack + 4 * iatt;   // xPack4 (k_pack_att4)
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    double q[4];
                    asm volatile("ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];"
                                 : "=d"(q[0]), "=d"(q[1]), "=d"(q[2]), "=d"(q[3])
                                 : "l"(xp + 4 * j));
#pragma unroll
                    for (int a = 0; a < 3; ++a) sum = fma(v[KT + 4 * a + j], q[a], sum);
                }
            }
#pragma unroll
            for (int j = 0; j < N_INSTR; ++j) sum = fma(v[KI + j], __ldg(xIns + c[j]), sum);
            if (NG > 0) sum = fma(v[NG > 0 ? KG : 0], xg, sum);
            if (NG < 0)
                for (int q = 0; q < A.nG; ++q) sum = fma(__ldcs(g + (KG + q) * TILE), __ldg(x + A.offGlob + q), sum);
            const double yi = fma(cy, y[i], cx * sum);
            y[i] = yi;
            sq = fma(yi, yi, sq);
        }
    }
    const double b = block_sum(sq, red);
    if (threadIdx.x == 0 && sqPartial) sqPartial[blockIdx.x] = b;
}

// ---------------------------------------------------------------------------------------
// aprod mode 2 (Eq. 3; Algorithm 3):  x <- cx*x + cy*(A^T y), one pass over A.
//   astro (Alg. 3 c.1-9; the paper uses atomicAdd): rows are sorted by star,
//     so each warp tile does a segmented inclusive scan over its 32 rows; a star whose rows lie
//     inside the tile is stored directly (single writer, no atomics); a star cut by a tile edge
//     leaves its partial in carryFirst/carryLast[tile] and k_astro_fixup adds the partials in
//     tile order -> bit-reproducible.
//   attitude and instrumental: RED.ADD.F64 to x, whose
//     att/instr/glob sections were pre-scaled by cx (k_scale).
//   gamma ("globSum1/globSum2"): warp -> CTA partial in fixed order, finished
//     by k_astro_fixup's extra block.
// SQUARE: terms are V^2 (y == 1): the column sums of squares of the preconditioner.
// coef = {cx, cy} in device memory.
// ---------------------------------------------------------------------------------------
// ATT_RED: scatter the attitude section here with REDs (fallback / preconditioner pass); when false
// the attitude section is done by k_aprod2_att on the time-ordered copy and the chunks of A that
// hold only attitude coefficients are not even loaded.
// PRIV ("shared-memory histogram plus global atomics", north_star): the CTA keeps private accumulators
// for the instrument columns [0, nInsSm) in shared memory (ATOMS, no L2 traffic) and only the other
// columns are added with REDs; the private table is flushed with one RED per touched column at the end.
// One CTA per SM (the table takes most of the shared memory).
#ifndef GSR_PRIV_THREADS
#define GSR_PRIV_THREADS 512
#endif
constexpr int PRIV_THREADS = GSR_PRIV_THREADS;   // fused pass (117 registers per thread)
// The standalone main kernel needs 64 registers: 32 warps per SM instead of 16 hide twice the load latency
// (Medium: 7.93 -> 6.86 ms)
constexpr int PRIV_THREADS_MAIN = 1024;
__host__ __device__ constexpr int priv_threads(bool fuse) { return fuse ? PRIV_THREADS : PRIV_THREADS_MAIN; }
// MATCH: sum the lanes of a warp that hit the same instrument column before the atomic (one MATCH.ANY per
// coefficient: costs 3.6 ms at Medium with uniform columns, saves 2.1 of 6.0 ms on the Zipf columns of Skewed;
// chosen per upload from the column histogram).
// FUSE (fused iteration, see k_combine_sumsq): before the scatter, the row's astro + instr + gamma terms of A*xin are
// added to yrw (which already holds cy*y + cx*(attitude terms)), the finished y_i is stored, its square summed
// into sqPartial, and y_i is the value that is scattered.
struct FuseArgs {
    const double *xin;     // operand of aprod1 (v), n doubles
    double *yrw;           // u, read-modify-write
    const double *coef1;   // {cx, cy} of aprod1
    double *sqPartial;     // per-CTA partial of sum y^2
    const double *xPack;   // FUSE_ATT: attitude unknowns of xin interleaved by axis (k_pack_att)
    cudaTextureObject_t texX;     // 0, or xin as a linear texture of int2 (gathers through the TEX path)
    cudaTextureObject_t texPack;  // 0, or xPack likewise
};
__device__ __forceinline__ double tex_f64(cudaTextureObject_t t, int64_t idx)
{
    const int2 q = tex1Dfetch<int2>(t, int(idx));
    return __hiloint2double(q.y, q.x);
}
// FUSE_ATT: the attitude terms of A*xin are gathered here too, in star order (whole aprod1 in this pass,
// y <- cy*y + cx*(A xin)); without it yrw must already hold cy*y + cx*(attitude terms).
// INS = false: the instrumental section is scattered by k_ins_scatter on the column-ordered copy instead (no atomics
// here, no shared-memory table, two CTAs of 256 threads per SM); without FUSE its coefficients and columns are not
// even loaded.
template <bool IC16, bool SQUARE, bool ATT_RED, bool PRIV = false, bool MATCH = false, bool FUSE = false, bool FUSE_ATT = false,
          bool INS = true, int NA = N_ASTRO, int NG = 1>
__global__ void __launch_bounds__(PRIV ? priv_threads(FUSE) : THREADS, PRIV ? 1 : 2)
k_aprod2(MatView A, const double *__restrict__ y, double *__restrict__ x,
         const double *__restrict__ coef, double *__restrict__ carryFirst,
         double *__restrict__ carryLast, double *__restrict__ globPartial, const int *done,
         FuseArgs F = FuseArgs{nullptr, nullptr, nullptr, nullptr, nullptr, 0, 0})
{
    __shared__ double red[32];
    __shared__ double gAcc[NG < 0 ? 32 : 1][NG < 0 ? MAX_GLOB : 1];   // NG = -1: per-warp sums of the global columns
    extern __shared__ double sIns[];   // PRIV: nInsSm private instrument accumulators
    if (done && *done) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    constexpr int PT = PRIV ? priv_threads(FUSE) : THREADS;
    const int nWarpsCta = PT / 32;
    const double cx = coef[0], cy = coef[1];
    const int64_t nTiles = (A.m + TILE - 1) / TILE;
    double *xAtt = x + A.offAtt;
    // instrumental REDs go to one of nRep replicas of the section (spreads the L2 atomic traffic
    // over nRep times more lines); k_astro_fixup folds the replicas into x in a fixed order
    double *xIns = A.insRep + int64_t((blockIdx.x * nWarpsCta + warp) % A.nRep) * A.nInstr;
    const int32_t nSm = PRIV ? A.nInsSm : 0;
    if (PRIV) {
        for (int c = threadIdx.x; c < nSm; c += PT) sIns[c] = 0.0;
        __syncthreads();
    }
    double gsum = 0.0, sq = 0.0;
    const double cx1 = FUSE ? F.coef1[0] : 0.0;
    const double xg1 = FUSE && NG > 0 ? __ldg(F.xin + A.offGlob) : 0.0;
    constexpr int KT = NA, KI = NA + N_ATT, KG = NA + N_ATT + N_INSTR, NP = KG + (NG > 0 ? NG : 0);
    const int np = NG < 0 ? A.nPar : NP;   // stored coefficients per row
    if (NG < 0) {
        if (lane < MAX_GLOB) gAcc[warp][lane] = 0.0;
        __syncwarp();
    }
    for (int64_t tile = int64_t(blockIdx.x) * nWarpsCta + warp; tile < nTiles;
         tile += int64_t(gridDim.x) * nWarpsCta) {
        const int64_t r0 = tile * TILE;
        const int nrows = int(min(int64_t(TILE), A.m - r0));
        const bool valid = lane < nrows;
        const int64_t i = r0 + (valid ? lane : nrows - 1);
        double v[NP];
        const double *g = A.V + tile * (int64_t(np) * TILE) + (valid ? lane : nrows - 1);
        load_row<ATT_RED || FUSE_ATT, INS || FUSE, NA, NG>(g, v);
        const unsigned long long tw = NA ? __ldg(A.tw + tile) : 0ull;   // one 8-byte word per tile: first star, head mask, cut flags
        const int64_t ia = NA ? NA * star_of(A, tw, i, valid ? lane : nrows - 1) : 0;
        // padded storage: the lanes past the last row read column 0 and a zero coefficient
        int32_t c[N_INSTR] = {0, 0, 0, 0, 0, 0};
        if (INS || FUSE) load_ic<IC16>(A, tile, lane, c);
        GSR_ASSERT(ia >= 0 && ia + NA <= A.offAtt);
#pragma unroll
        for (int j = 0; j < N_INSTR; ++j) GSR_ASSERT(c[j] >= 0 && c[j] < A.nInstr);
        double yv = 0.0;
        if (FUSE) {
            if (valid) {
                const double *xa = F.xin + ia, *xIn = F.xin + A.offInstr;
                double sum = 0.0;
#pragma unroll
                for (int k = 0; k < NA; ++k) sum = fma(v[k], __ldg(xa + k), sum);
#pragma unroll
                for (int j = 0; j < N_INSTR; ++j) {
                    const double xj = F.texX ? tex_f64(F.texX, A.offInstr + c[j]) : __ldg(xIn + c[j]);
                    sum = fma(v[KI + j], xj, sum);
                }
                if (NG > 0) sum = fma(v[NG > 0 ? KG : 0], xg1, sum);
                if (NG < 0)
                    for (int q = 0; q < A.nG; ++q) sum = fma(__ldg(g + (KG + q) * TILE), __ldg(F.xin + A.offGlob + q), sum);
                double yOld = F.yrw[i];
                if (FUSE_ATT) {
                    const int64_t iattRow = __ldcs(A.iatt + i);
                    GSR_ASSERT(iattRow >= 0 && iattRow + 4 <= A.nDof);
                    const double *xp = F.xPack + 3 * iattRow;
#pragma unroll
                    for (int j = 0; j < 4; ++j)
#pragma unroll
                        for (int a = 0; a < 3; ++a) {
                            const double xa3 = F.texPack ? tex_f64(F.texPack, 3 * iattRow + 3 * j + a) : __ldg(xp + 3 * j + a);
                            sum = fma(v[KT + 4 * a + j], xa3, sum);
                        }
                    yOld *= F.coef1[1];
                }
                const double yi = fma(cx1, sum, yOld);
                F.yrw[i] = yi;
                sq = fma(yi, yi, sq);
                yv = cy * yi;
            }
        } else if (valid) {
            yv = SQUARE ? 1.0 : cy * y[i];
        }
#pragma unroll
        for (int k = 0; k < NP; ++k) v[k] = SQUARE ? v[k] * v[k] * yv : v[k] * yv;

        // ---- attitude + instrumental scatter (invalid lanes hold zeros and add nothing)
        if (ATT_RED && valid) {
            GSR_ASSERT(A.iatt[i] >= 0 && A.iatt[i] + 4 <= A.nDof);
            double *xt = xAtt + A.iatt[i];
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int j = 0; j < 4; ++j) atomicAdd(xt + a * A.nDof + j, v[KT + 4 * a + j]);
        }
        if (INS) {
#pragma unroll
            for (int j = 0; j < N_INSTR; ++j) {
                // lanes of the warp that hit the same column (hot columns of a skewed distribution) are summed
                // in lane order first and the lowest lane adds once: no same-address atomics inside a warp
                double val = v[KI + j];
                bool add = valid;
                const unsigned peers = MATCH ? __match_any_sync(0xffffffffu, valid ? c[j] : -1 - lane) : 0u;
                if (MATCH && __any_sync(0xffffffffu, (peers & (peers - 1)) != 0)) {
                    const int n = __reduce_max_sync(0xffffffffu, __popc(peers));
                    unsigned p = peers;
                    double sum = 0.0;
                    for (int it = 0; it < n; ++it) {
                        const int src = p ? __ffs(p) - 1 : lane;
                        const double t = __shfl_sync(0xffffffffu, val, src);
                        if (p) sum += t;
                        p &= p - 1;
                    }
                    val = sum;
                    add = valid && lane == __ffs(peers) - 1;
                }
                if (add) {
                    if (PRIV && c[j] < nSm) atomicAdd(sIns + c[j], val);
                    else atomicAdd(xIns + c[j], val);
                }
            }
        }
        // ---- gamma: fixed-order warp sum, accumulated per warp over its tiles
        if (NG > 0) gsum += v[NG > 0 ? KG : 0];   // per lane over its tiles; the lanes are summed once, after the loop
        if (NG < 0) {   // every global column: fixed-order warp sum into this warp's accumulator (lanes past the last row: yv = 0)
            for (int q = 0; q < A.nG; ++q) {
                const double a = __ldg(g + (KG + q) * TILE);
                const double t = warp_sum(SQUARE ? a * a * yv : a * yv);
                if (lane == 0) gAcc[warp][q] += t;
            }
        }

        // ---- astro: segmented scan by star over the tile's rows
        if (NA == 0) continue;
        const unsigned heads = uint32_t(tw) | 1u;          // segment starts inside the tile (lane 0 always opens one)
        if (heads == 1u) {   // the whole tile belongs to one star (the common case): totals instead of a scan
            double s5[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll
            for (int k = 0; k < NA; ++k) s5[k] = v[k];
            const double tot = warp_sum5(s5, lane);
            const int k = (lane >> 2) & 7;   // lane 4k holds value k
            if ((lane & 3) == 0 && k < NA) {
                // the star began in an earlier tile and / or goes on in the next one: the fix-up adds the pieces
                if (!(uint32_t(tw) & 1u) || ((tw >> 61) & 1ull)) carryFirst[tile * N_ASTRO + k] = tot;
                else x[ia + k] = fma(cx, x[ia + k], tot);
            }
            continue;
        }
        const bool tail = valid && ((lane == nrows - 1) || ((heads >> 1) >> lane) & 1u);
        const int segStart = 31 - __clz(heads & (0xffffffffu >> (31 - lane)));
        const int dist = lane - segStart;
        double s[NA > 0 ? NA : 1];
#pragma unroll
        for (int k = 0; k < NA; ++k) s[k] = v[k];
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
#pragma unroll
            for (int k = 0; k < NA; ++k) {
                const double t = __shfl_up_sync(0xffffffffu, s[k], d);
                if (dist >= d) s[k] += t;
            }
        }
        if (tail) {
            bool cut = false;
            if (segStart == 0) cut = !(uint32_t(tw) & 1u);            // the star began in an earlier tile
            if (lane == nrows - 1) cut = cut || ((tw >> 61) & 1ull);   // and / or goes on in the next one
            if (!cut) {
                double *xa = x + ia;
#pragma unroll
                for (int k = 0; k < NA; ++k) xa[k] = fma(cx, xa[k], s[k]);
            } else {
                GSR_ASSERT(tile >= 0 && tile < nTiles);
                double *c = (segStart == 0 ? carryFirst : carryLast) + tile * N_ASTRO;
#pragma unroll
                for (int k = 0; k < NA; ++k) c[k] = s[k];
            }
        }
    }
    // CTA partial of gamma in fixed order: every lane summed its own rows in tile order, then a fixed tree over the lanes and
    // the warps in order
    if (NG > 0) gsum = warp_sum(gsum);
    __syncthreads();
    if (lane == 0) red[warp] = gsum;
    __syncthreads();
    if (NG > 0 && threadIdx.x == 0) {
        double g = 0.0;
        for (int w = 0; w < nWarpsCta; ++w) g += red[w];
        globPartial[blockIdx.x] = g;
    }
    if (NG < 0 && threadIdx.x < A.nG) {   // globPartial[q*gridDim.x + blockIdx.x]: this CTA's share of global column q
        double g = 0.0;
        for (int w = 0; w < nWarpsCta; ++w) g += gAcc[w][threadIdx.x];
        globPartial[int64_t(threadIdx.x) * gridDim.x + blockIdx.x] = g;
    }
    if (FUSE) {
        const double b = block_sum(sq, red);
        if (threadIdx.x == 0) F.sqPartial[blockIdx.x] = b;
    }
    if (PRIV) {   // flush the private table (the barrier above ordered the ATOMS before these reads)
        for (int c = threadIdx.x; c < nSm; c += PT) {
            const double t = sIns[c];
            if (t != 0.0) atomicAdd(xIns + c, t);
        }
    }
}

// Finishes the astro section (stars cut by tile edges, stars without rows) and gamma.
// One thread per star; the last block sums the gamma partials.  Deterministic.
__global__ void __launch_bounds__(256)
k_astro_fixup(MatView A, double *__restrict__ x, const double *__restrict__ coef,
              const double *__restrict__ carryFirst, const double *__restrict__ carryLast,
              const double *__restrict__ globPartial, int nGlobPartial, const int *done)
{
    __shared__ double red[32];
    if (done && *done) return;
    const double cx = coef[0];
    const int starBlocks = A.nA > 0 ? int((A.nStars + blockDim.x - 1) / blockDim.x) : 0;
    if (blockIdx.x == gridDim.x - 1) {
        for (int q = 0; q < A.nG; ++q) {
            double g = 0.0;
            for (int p = threadIdx.x; p < nGlobPartial; p += blockDim.x) g += globPartial[int64_t(q) * nGlobPartial + p];
            g = block_sum(g, red);
            if (threadIdx.x == 0) x[A.offGlob + q] += g;   // section already scaled by cx
        }
        return;
    }
    if (blockIdx.x >= starBlocks) {
        // fold the instrument replicas (replica order fixed) into the pre-scaled section
        const int64_t c = int64_t(blockIdx.x - starBlocks) * blockDim.x + threadIdx.x;
        if (c < A.nInstr) {
            double t = 0.0;
            for (int r = 0; r < A.nRep; ++r) t += A.insRep[int64_t(r) * A.nInstr + c];
            x[A.offInstr + c] += t;
        }
        return;
    }
    const int64_t s = int64_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (s >= A.nStars) return;
    const int64_t r0 = A.rp[s], r1 = A.rp[s + 1];
    GSR_ASSERT(r0 >= 0 && r0 <= r1 && r1 <= A.m);
    double *xa = x + s * A.nA;
    if (r0 == r1) {
        for (int k = 0; k < A.nA; ++k) xa[k] *= cx;
        return;
    }
    const int64_t t0 = r0 / TILE, t1 = (r1 - 1) / TILE;
    if (t0 == t1) return;   // stored by k_aprod2
    double acc[N_ASTRO] = {0, 0, 0, 0, 0};
    for (int64_t t = t0; t <= t1; ++t) {
        const double *c = ((t == t0 && r0 != t * TILE) ? carryLast : carryFirst) + t * N_ASTRO;
#pragma unroll
        for (int k = 0; k < N_ASTRO; ++k) acc[k] += k < A.nA ? c[k] : 0.0;
    }
#pragma unroll
    for (int k = 0; k < N_ASTRO; ++k)
        if (k < A.nA) xa[k] = fma(cx, xa[k], acc[k]);
}

// Before the scatter of aprod2: x[lo..hi) *= coef[0] (att + instr + gamma sections, only when
// prescale) and the instrument replicas are zeroed.
__global__ void k_pre_aprod2(double *__restrict__ x, int64_t lo, int64_t hi,
                             const double *__restrict__ coef, double *__restrict__ rep,
                             int64_t nRepTotal, int prescale, const int *done)
{
    if (done && *done) return;
    const int64_t tid = int64_t(blockIdx.x) * blockDim.x + threadIdx.x;
    const int64_t nth = int64_t(gridDim.x) * blockDim.x;
    if (prescale == 2) {   // plain zero fill (the buffer may hold anything)
        for (int64_t j = lo + tid; j < hi; j += nth) x[j] = 0.0;
    } else if (prescale) {
        const double c = coef[0];
        for (int64_t j = lo + tid; j < hi; j += nth) x[j] *= c;
    }
    for (int64_t j = tid; j < nRepTotal; j += nth) rep[j] = 0.0;
}

// ---------------------------------------------------------------------------------------
// aprod2, attitude section on the time-ordered copy ("bucketed scatter", north_star; the
// paper's kernels use one atomicAdd per coefficient, Alg. 3).  Rows t are
// sorted by attitude start s, so the 32 rows of a warp tile share very few distinct s: a
// segmented scan by s over the tile leaves one sum per (s, axis, j) and only those are added to x
// (RED), instead of 12 REDs per row.  y is gathered through permT (one 8-byte gather per row).
// ---------------------------------------------------------------------------------------
// LINEAR: y is already in block-time order (the uT copy written by the fused pass): no permT, no gather, no prefetch.
template <bool SQUARE, bool LINEAR = false>
__global__ void __launch_bounds__(256)
k_aprod2_att(MatView A, const double *__restrict__ y, double *__restrict__ x,
             const double *__restrict__ coef, const int *done)
{
    if (done && *done) return;
    const int lane = threadIdx.x & 31;
    const double cy = coef[1];
    double *xAtt = x + A.offAtt;
    const int64_t nTiles = (A.m + TILE - 1) / TILE;
    const int64_t warpId = (int64_t(blockIdx.x) * blockDim.x + threadIdx.x) >> 5;
    const int64_t nWarps = (int64_t(gridDim.x) * blockDim.x) >> 5;
    for (int64_t tile = warpId; tile < nTiles; tile += nWarps) {
        const int64_t t0 = tile * TILE;
        const int nrows = int(min(int64_t(TILE), A.m - t0));
        const bool valid = lane < nrows;
        const int64_t t = t0 + (valid ? lane : nrows - 1);
        const int32_t sv = __ldcs(A.sT + t);
        GSR_ASSERT(sv >= 0 && int64_t(sv) + 4 <= A.nDof && (LINEAR || SQUARE || int64_t(A.permT[t]) < A.m));
        // The gathers below land anywhere in this block's slice of y.  Pull the NEXT block's slice
        // into L2 linearly while this block is processed (one 32-byte sector per 4 rows): first touches
        // that arrive together are not merged by L2 and would each go to DRAM (measured).
        if (!SQUARE && !LINEAR && (lane & 3) == 0 && t + (int64_t(1) << ATT_BLOCK_BITS) < A.m)
            asm volatile("prefetch.global.L2 [%0];" ::"l"(y + t + (int64_t(1) << ATT_BLOCK_BITS)));
        double yv = 0.0;
        if (valid) yv = SQUARE ? 1.0 : cy * (LINEAR ? __ldcs(y + t) : __ldg(y + __ldcs(A.permT + t)));
        double v[N_ATT];
#pragma unroll
        for (int k = 0; k < N_ATT; ++k) {
            const double a = __ldcs(A.attT + int64_t(k) * A.m + t);
            v[k] = SQUARE ? a * a * yv : a * yv;
        }
        const int32_t sPrev = __shfl_up_sync(0xffffffffu, sv, 1);
        const int32_t sNext = __shfl_down_sync(0xffffffffu, sv, 1);
        const bool head = (lane == 0) || (sv != sPrev);
        const bool tail = valid && ((lane == nrows - 1) || (sv != sNext));
        const unsigned heads = __ballot_sync(0xffffffffu, head);
        if (heads == 1u) {
            // one s in the whole tile (the common case): plain warp sums, lanes 0..11 add one each
            double mine = 0.0;
#pragma unroll
            for (int k = 0; k < N_ATT; ++k) {
                const double t2 = warp_sum(v[k]);
                if (lane == k) mine = t2;
            }
            if (lane < N_ATT) atomicAdd(xAtt + int64_t(lane >> 2) * A.nDof + sv + (lane & 3), mine);
        } else {
            const int segStart = 31 - __clz(heads & (0xffffffffu >> (31 - lane)));
            const int dist = lane - segStart;
            // scan steps only up to the longest segment of this tile (segments are short when the
            // block holds few rows per attitude start)
            const int maxDist = __reduce_max_sync(0xffffffffu, dist);
            for (int d = 1; d <= maxDist; d <<= 1) {
#pragma unroll
                for (int k = 0; k < N_ATT; ++k) {
                    const double t2 = __shfl_up_sync(0xffffffffu, v[k], d);
                    if (dist >= d) v[k] += t2;
                }
            }
            if (tail) {
#pragma unroll
                for (int a = 0; a < 3; ++a)
#pragma unroll
                    for (int j = 0; j < 4; ++j) atomicAdd(xAtt + a * A.nDof + sv + j, v[4 * a + j]);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------
// aprod2, instrumental section on the column-ordered copy (Alg. 3 instr; the paper uses one atomicAdd
// per coefficient).  Rows are cut into blocks of INS_BLOCK and the 6 x INS_BLOCK coefficients of a block are sorted by
// column; the columns are cut into insNB buckets of insW <= INS_BUCKET_MAX.  CTA (g, k) keeps the accumulators of
// bucket k in shared memory for its whole life and walks the row blocks g, g + nG, ...: it stages the block's slice of
// y through L1 (32 KB), streams the bucket's entries (12 bytes each, coalesced), multiplies with the gathered y, sums equal columns with a warp segmented scan (they are adjacent) and adds the sum to the
// accumulator with a plain read-modify-write: a column whose entries lie inside one 32-entry chunk belongs to that
// chunk alone; only the first and last column of a chunk can continue in a neighbour chunk and take a shared-memory
// atomic.  (y: see the kernel; a first version staged the slice in shared memory behind two barriers per block and ran
// at 1.1 TB/s, bound by the latency of those phases.)  No global atomics: every CTA writes its table to its own slice of insRep and k_astro_fixup folds the slices
// in a fixed order.  The eight CTAs of a group read the same slice of y at about the same time (L2).
// ---------------------------------------------------------------------------------------
constexpr int INS_THREADS = 1024;    // k_ins_scatter: 32 warps, one CTA per SM
constexpr int INS_WARPS = INS_THREADS / 32;   // a bucket is cut into INS_WARPS sub-buckets, one per warp
constexpr int INS_UNROLL = 8;        // 32-entry chunks of a sub-bucket that a warp holds in registers
// streaming loads that do not displace anything in L1
__device__ __forceinline__ uint32_t ld_stream_u32(const uint32_t *p)
{
    uint32_t v;
    asm volatile("ld.global.nc.L1::no_allocate.u32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ double ld_stream_f64(const double *p)
{
    double v;
    asm volatile("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
__global__ void __launch_bounds__(INS_THREADS, 1)
k_ins_scatter(MatView A, const double *__restrict__ y, const double *__restrict__ coef, const int *done)
{
    extern __shared__ double sIns[];   // [insW] accumulators of this CTA's column bucket, then 2 x [INS_BLOCK] slices of y
    if (done && *done) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int k = blockIdx.x % A.insNB, g = blockIdx.x / A.insNB, nG = gridDim.x / A.insNB;
    if (g >= nG) return;
    const int c0 = k * A.insW, w = max(0, min(A.insW, int(A.nInstr) - c0));
    double *acc = sIns - c0;           // indexed by the column itself
    double *ybuf = sIns + A.insW;
    const double cy = coef[1];
    for (int c = threadIdx.x; c < A.insW; c += INS_THREADS) sIns[c] = 0.0;
    const int64_t nBlocks = (A.m + INS_BLOCK - 1) >> INS_ROW_BITS;
    const int nSub = A.insNB * INS_WARPS;
    const int64_t *ptr = A.insPtr + k * INS_WARPS + warp;   // + b*nSub: this warp's sub-bucket of block b

    // the block's slice of y, copied to shared memory one block ahead (8-byte cp.async: no alignment demands on y)
    auto stage = [&](int64_t b, int buf) {
        if (b < nBlocks) {
            const int64_t r0 = b << INS_ROW_BITS;
            const int nr = int(min(int64_t(INS_BLOCK), A.m - r0));
            const unsigned dst = unsigned(__cvta_generic_to_shared(ybuf + buf * INS_BLOCK));
            for (int r = threadIdx.x; r < nr; r += INS_THREADS)
                asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst + 8u * r), "l"(y + r0 + r));
        }
        asm volatile("cp.async.commit_group;");
    };
    // one 32-entry chunk: sums of equal (adjacent) columns, then one plain read-modify-write per column: the columns of a
    // sub-bucket belong to this warp alone
    auto chunk = [&](uint32_t meta, double val, bool valid, const double *yb) {
        const int col = int(meta >> INS_ROW_BITS);
        GSR_ASSERT(!valid || (col >= c0 && col < c0 + w));
        double s = valid ? val * (cy * yb[meta & (INS_BLOCK - 1)]) : 0.0;
        // segmented inclusive scan by column, two fixed steps (runs of up to 4 equal columns); longer runs take more steps
        // (every lane takes part in every shuffle: no shuffle on the right of a short-circuit operator)
        const int up1 = __shfl_up_sync(0xffffffffu, col, 1), up2 = __shfl_up_sync(0xffffffffu, col, 2);
        const int up4 = __shfl_up_sync(0xffffffffu, col, 4), dn1 = __shfl_down_sync(0xffffffffu, col, 1);
        const bool p1 = lane >= 1 && col == up1;
        const bool p2 = lane >= 2 && col == up2;
        const bool tail = valid && (lane == 31 || col != dn1);
        double t = __shfl_up_sync(0xffffffffu, s, 1);
        if (p1) s += t;
        t = __shfl_up_sync(0xffffffffu, s, 2);
        if (p2) s += t;
        if (__any_sync(0xffffffffu, lane >= 4 && col == up4)) {
            for (int d = 4; d < 32; d <<= 1) {
                const int upd = __shfl_up_sync(0xffffffffu, col, d);
                t = __shfl_up_sync(0xffffffffu, s, d);
                if (lane >= d && col == upd) s += t;
            }
        }
        if (tail) acc[col] += s;
        __syncwarp();   // a column that goes on in the next chunk is read-modify-written again by another lane
    };

    // The first INS_UNROLL chunks of the sub-bucket live in registers and are loaded one block ahead: chunk q of the next
    // block is requested as soon as chunk q of this block is done (more than INS_UNROLL chunks is rare; the rest is loaded
    // when its turn comes).
    uint32_t meta[INS_UNROLL];
    double val[INS_UNROLL];
    int64_t e0 = 0;
    int cnt = 0;
    if (g < nBlocks) {
        e0 = __ldg(ptr + int64_t(g) * nSub);
        cnt = int(__ldg(ptr + int64_t(g) * nSub + 1) - e0);
    }
    {
        const uint32_t *mp = A.insMeta + e0 + lane;
        const double *vp = A.insVal + e0 + lane;
#pragma unroll
        for (int q = 0; q < INS_UNROLL; ++q) {
            const bool valid = q * 32 + lane < cnt;
            meta[q] = valid ? ld_stream_u32(mp + q * 32) : (0xffffffffu - lane);   // past the end: distinct columns
            val[q] = valid ? ld_stream_f64(vp + q * 32) : 0.0;
        }
    }
    stage(g, 0);
    int buf = 0;
    for (int64_t b = g; b < nBlocks; b += nG, buf ^= 1) {
        int64_t e0n = 0;
        int cntn = 0;
        if (b + nG < nBlocks) {
            e0n = __ldg(ptr + (b + nG) * nSub);
            cntn = int(__ldg(ptr + (b + nG) * nSub + 1) - e0n);
        }
        asm volatile("cp.async.wait_group 0;");
        __syncthreads();   // this block's slice of y has landed, and every warp is done with the other buffer
        stage(b + nG, buf ^ 1);
        const double *yb = ybuf + buf * INS_BLOCK;
        const uint32_t *mp = A.insMeta + e0n + lane;
        const double *vp = A.insVal + e0n + lane;
#pragma unroll
        for (int q = 0; q < INS_UNROLL; ++q) {
            if (q * 32 < cnt) chunk(meta[q], val[q], q * 32 + lane < cnt, yb);   // warp-uniform condition
            const bool valid = q * 32 + lane < cntn;
            meta[q] = valid ? ld_stream_u32(mp + q * 32) : (0xffffffffu - lane);
            val[q] = valid ? ld_stream_f64(vp + q * 32) : 0.0;
        }
        for (int o = 32 * INS_UNROLL; o < cnt; o += 32) {   // overflow of the register window
            const bool valid = o + lane < cnt;
            const uint32_t mt = valid ? ld_stream_u32(A.insMeta + e0 + o + lane) : (0xffffffffu - lane);
            const double vl = valid ? ld_stream_f64(A.insVal + e0 + o + lane) : 0.0;
            chunk(mt, vl, valid, yb);
        }
        e0 = e0n;
        cnt = cntn;
    }
    asm volatile("cp.async.wait_group 0;");
    __syncthreads();
    double *out = A.insRep + int64_t(g) * A.nInstr + c0;
    for (int c = threadIdx.x; c < w; c += INS_THREADS) out[c] = sIns[c];
}

// Build of the column-ordered copy (setup).  key = block << INS_KEY_BLOCK | column << INS_KEY_COL | row in block << 3 | slot for the 6
// coefficients of rows [row0, row0 + cnt); a keys-only radix sort (cub) orders them; k_ins_fill turns the sorted keys
// into insMeta / insVal; k_ins_ptr finds the first entry of every (block, bucket).
__global__ void k_ins_keys(MatView A, int64_t row0, int64_t cnt, unsigned long long *__restrict__ key)
{
    for (int64_t q = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; q < cnt * N_INSTR; q += int64_t(gridDim.x) * blockDim.x) {
        const int64_t i = row0 + q / N_INSTR;
        const int j = int(q % N_INSTR);
        const unsigned long long col = (unsigned long long)ic_at(A, cpos(i, j));
        key[q] = ((unsigned long long)(i >> INS_ROW_BITS) << INS_KEY_BLOCK) | (col << INS_KEY_COL) | ((unsigned long long)(i & (INS_BLOCK - 1)) << 3) |
                 (unsigned long long)j;
    }
}
__global__ void k_ins_fill(MatView A, int64_t e0, int64_t cnt, const unsigned long long *__restrict__ key,
                           uint32_t *__restrict__ meta)
{
    for (int64_t q = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; q < cnt; q += int64_t(gridDim.x) * blockDim.x) {
        const unsigned long long kk = key[q];
        const int64_t i = (int64_t(kk >> INS_KEY_BLOCK) << INS_ROW_BITS) | int64_t((kk >> 3) & (INS_BLOCK - 1));
        meta[e0 + q] = (uint32_t((kk >> INS_KEY_COL) & 0xffffu) << INS_ROW_BITS) | uint32_t((kk >> 3) & (INS_BLOCK - 1));
        A.insVal[e0 + q] = A.V[vpos(i, N_ASTRO + N_ATT + int(kk & 7))];
    }
}
// insPtr[b*nSub + j] = first entry e of block b with column >= j*(insW/INS_WARPS), nSub = insNB*INS_WARPS sub-buckets
// (entries of block b start at 6*b*INS_BLOCK)
__global__ void k_ins_ptr(MatView A, int64_t *__restrict__ ptr)
{
    const int64_t nBlocks = (A.m + INS_BLOCK - 1) >> INS_ROW_BITS;
    const int nSub = A.insNB * INS_WARPS, ws = A.insW / INS_WARPS;
    for (int64_t q = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; q <= nBlocks * nSub; q += int64_t(gridDim.x) * blockDim.x) {
        if (q == nBlocks * nSub) {
            ptr[q] = A.m * N_INSTR;
            continue;
        }
        const int64_t b = q / nSub;
        const uint32_t colLo = uint32_t(q % nSub) * uint32_t(ws);
        int64_t lo = b * (int64_t(INS_BLOCK) * N_INSTR), hi = min(A.m, (b + 1) << INS_ROW_BITS) * N_INSTR;
        while (lo < hi) {
            const int64_t mid = (lo + hi) >> 1;
            if ((A.insMeta[mid] >> INS_ROW_BITS) < colLo) lo = mid + 1; else hi = mid;
        }
        ptr[q] = lo;
    }
}
// After the preconditioner: the copy takes the same factors as the row layout (same operands, bit-identical values)
__global__ void k_scale_ins(MatView A, const double *__restrict__ p)
{
    for (int64_t e = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; e < A.m * N_INSTR; e += int64_t(gridDim.x) * blockDim.x)
        A.insVal[e] = A.insVal[e] * p[A.offInstr + (A.insMeta[e] >> INS_ROW_BITS)];
}

// ---------------------------------------------------------------------------------------
// Fused LSQR iteration (gsr_lsqr uses it when the attitude copy exists; constraint rows keep
// their own two kernels): u' = A v - alpha u is row-local and A^T is linear, so the astro / instr / gamma sections of
// t = A^T u' are accumulated, unscaled, by the star-ordered pass that computes u' (k_aprod2<.., FUSE, FUSE_ATT>:
// the whole of aprod1 plus the scatter of aprod2's main kernel on one read of A); k_aprod2_att adds the
// attitude section of t; then v <- cxv*v + cyv*t with sum v^2 (k_combine_sumsq), which applies 1/beta.
// Per iteration 248 + 112 B/row are streamed instead of 248 + 136 + 112.
// ---------------------------------------------------------------------------------------
// v <- c[0]*v + c[1]*t and the per-CTA partial of sum v^2 (fixed order for a fixed grid)
__global__ void __launch_bounds__(256)
k_combine_sumsq(double *__restrict__ v, const double *__restrict__ t, int64_t n, const double *__restrict__ coef,
                double *__restrict__ partial, const int *done)
{
    __shared__ double red[32];
    if (done && *done) return;
    const double cv = coef[0], ct = coef[1];
    double s = 0.0;
    for (int64_t j = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; j < n;
         j += int64_t(gridDim.x) * blockDim.x) {
        const double r = fma(cv, v[j], ct * t[j]);
        v[j] = r;
        s = fma(r, r, s);
    }
    s = block_sum(s, red);
    if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

// attT[k*m + t] = V[permT[t]*24 + 5 + k]  (at upload; k_scale_attT applies the preconditioner to the copy)
__global__ void k_gather_att(MatView A)
{
    for (int64_t t = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; t < A.m;
         t += int64_t(gridDim.x) * blockDim.x) {
        const int64_t i = A.permT[t];
#pragma unroll
        for (int k = 0; k < N_ATT; ++k) A.attT[int64_t(k) * A.m + t] = A.V[vpos(i, A.nA + k, A.nPar)];
    }
}

// After the preconditioner: the copy takes the same factors as the row layout, attT[k][t] *= p[column of (t, k)]
// (same operands as k_scale_values, so the two stay bit-identical), coalesced instead of a second gather.
__global__ void k_scale_attT(MatView A, const double *__restrict__ p)
{
    for (int64_t t = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; t < A.m;
         t += int64_t(gridDim.x) * blockDim.x) {
        const double *pc = p + A.offAtt + A.sT[t];
#pragma unroll
        for (int kk = 0; kk < N_ATT; ++kk) {
            const int64_t e = int64_t(kk) * A.m + t;
            A.attT[e] = A.attT[e] * pc[(kk >> 2) * A.nDof + (kk & 3)];
        }
    }
}

// uT[t] = u[permT[t]]: u^ brought into block-time order for k_aprod2_att<.., LINEAR>.  A pass of its own: the gather
// (inside the block's 16 MB slice of u, pulled into L2 linearly one block ahead as in k_aprod2_att) runs with far more
// parallelism here than as a dependent step of the attitude kernel, and the writes are coalesced.
__global__ void __launch_bounds__(256)
k_u_to_time(const double *__restrict__ u, const uint32_t *__restrict__ permT, int64_t m, double *__restrict__ uT,
            const int *done)
{
    if (done && *done) return;
    // one row per thread: four rows per thread with the gathers batched ran 2 ms slower (the gathers then outrun the
    // linear prefetch of the next block and their first touches go to DRAM one by one)
    for (int64_t t = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; t < m; t += int64_t(gridDim.x) * blockDim.x) {
        if ((t & 3) == 0 && t + (int64_t(1) << ATT_BLOCK_BITS) < m)
            asm volatile("prefetch.global.L2 [%0];" ::"l"(u + t + (int64_t(1) << ATT_BLOCK_BITS)));
        GSR_ASSERT(int64_t(permT[t]) < m);
        uT[t] = __ldg(u + __ldcs(permT + t));
    }
}

// keys / values of the time sort of rows [i0, i0+cnt): key = attitude start (int32), value = row
__global__ void k_sort_keys(const int32_t *__restrict__ iatt, int64_t i0, int64_t cnt, int32_t *__restrict__ key,
                            uint32_t *__restrict__ val)
{
    for (int64_t q = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; q < cnt;
         q += int64_t(gridDim.x) * blockDim.x) {
        key[q] = iatt[i0 + q];
        val[q] = uint32_t(i0 + q);
    }
}

// ---------------------------------------------------------------------------------------
// Model variants.  PAPER.md:78 allows 0 <= N_Astro <= 5 astrometric and 0 <= N_Instr <= 6
// instrumental coefficients per row and runs with or without the global part; the paper also ran 5 global
// parameters, and its 40 / 100 / 300 GB datasets solve only some of the sections.
// These two kernels compute the same products (Eq. 2-3, Alg. 2-3) for any such layout: the section widths are
// read from MatView at run time, every coefficient is loaded where it is used (coalesced, tile-transposed storage
// of width nPar) and nothing is kept in per-thread arrays.  The 5/12/6/1 production layout keeps its specialised
// kernels above.  aprod2: astro by the same segmented scan (no atomics, carries for stars cut by a tile edge),
// attitude and instrumental by RED.ADD.F64, every global column by warp sum -> per-warp shared-memory
// accumulator -> CTA partial -> k_fixup_gen (fixed order).
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(THREADS)
k_aprod1_gen(MatView A, const double *__restrict__ x, double *__restrict__ y, const double *__restrict__ coef,
             double *__restrict__ sqPartial, const int *done)
{
    __shared__ double red[32];
    if (done && *done) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const double cx = coef[0], cy = coef[1];
    const int64_t nTiles = (A.m + TILE - 1) / TILE;
    const int kT = A.nA + A.nAtt, kI = kT + A.nI;
    double sq = 0.0;
    for (int64_t tile = int64_t(blockIdx.x) * WARPS + warp; tile < nTiles; tile += int64_t(gridDim.x) * WARPS) {
        const int64_t r0 = tile * TILE;
        const int nrows = int(min(int64_t(TILE), A.m - r0));
        if (lane < nrows) {
            const int64_t i = r0 + lane;
            const double *g = A.V + tile * (int64_t(A.nPar) * TILE) + lane;
            double sum = 0.0;
            if (A.nA > 0) {
                const double *xa = x + A.nA * star_of(A, __ldg(A.tw + tile), i, lane);
                GSR_ASSERT(xa >= x && xa + A.nA <= x + A.offAtt);
                for (int k = 0; k < A.nA; ++k) sum = fma(__ldcs(g + k * TILE), __ldg(xa + k), sum);
            }
            if (A.nAtt > 0) {
                const int64_t s = __ldcs(A.iatt + i);
                GSR_ASSERT(s >= 0 && s + 4 <= A.nDof);
                const double *xt = x + A.offAtt + s;
#pragma unroll
                for (int a = 0; a < 3; ++a)
#pragma unroll
                    for (int j = 0; j < 4; ++j)
                        sum = fma(__ldcs(g + (A.nA + 4 * a + j) * TILE), __ldg(xt + a * A.nDof + j), sum);
            }
            for (int j = 0; j < A.nI; ++j) {
                const int32_t c = ic_at(A, (tile * A.nI + j) * TILE + lane);
                GSR_ASSERT(c >= 0 && c < A.nInstr);
                sum = fma(__ldcs(g + (kT + j) * TILE), __ldg(x + A.offInstr + c), sum);
            }
            for (int q = 0; q < A.nG; ++q) sum = fma(__ldcs(g + (kI + q) * TILE), __ldg(x + A.offGlob + q), sum);
            const double yi = fma(cy, y[i], cx * sum);
            y[i] = yi;
            sq = fma(yi, yi, sq);
        }
    }
    const double b = block_sum(sq, red);
    if (threadIdx.x == 0 && sqPartial) sqPartial[blockIdx.x] = b;
}

// x <- cx*x + cy*(A^T y); the attitude / instrumental / global sections of x were multiplied by cx beforehand
// (k_pre_aprod2).  globPartial[q*gridDim.x + blockIdx.x]: this CTA's share of global column q.
// ATT = false: the attitude section is left to k_aprod2_att on the block-time-ordered copy (which does not depend on the
// other sections' widths).
template <bool SQUARE, bool ATT = true>
__global__ void __launch_bounds__(THREADS)
k_aprod2_gen(MatView A, const double *__restrict__ y, double *__restrict__ x, const double *__restrict__ coef,
             double *__restrict__ carryFirst, double *__restrict__ carryLast, double *__restrict__ globPartial,
             const int *done)
{
    __shared__ double gAcc[WARPS][MAX_GLOB];
    if (done && *done) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const double cx = coef[0], cy = coef[1];
    const int64_t nTiles = (A.m + TILE - 1) / TILE;
    const int kT = A.nA + A.nAtt, kI = kT + A.nI;
    if (lane < MAX_GLOB) gAcc[warp][lane] = 0.0;
    __syncwarp();
    for (int64_t tile = int64_t(blockIdx.x) * WARPS + warp; tile < nTiles; tile += int64_t(gridDim.x) * WARPS) {
        const int64_t r0 = tile * TILE;
        const int nrows = int(min(int64_t(TILE), A.m - r0));
        const bool valid = lane < nrows;
        const int ln = valid ? lane : nrows - 1;
        const int64_t i = r0 + ln;
        const double *g = A.V + tile * (int64_t(A.nPar) * TILE) + ln;
        const double yv = valid ? (SQUARE ? 1.0 : cy * y[i]) : 0.0;     // lanes past the last row add zeros
        if (A.nA > 0) {   // ---- astro: segmented scan by star, as in k_aprod2
            const unsigned long long tw = __ldg(A.tw + tile);
            const int64_t ia = A.nA * star_of(A, tw, i, ln);
            GSR_ASSERT(ia >= 0 && ia + A.nA <= A.offAtt);
            const unsigned heads = uint32_t(tw) | 1u;
            const bool tail = valid && ((lane == nrows - 1) || ((heads >> 1) >> lane) & 1u);
            const int segStart = 31 - __clz(heads & (0xffffffffu >> (31 - lane)));
            const int dist = lane - segStart;
            bool cut = false;
            if (segStart == 0) cut = !(uint32_t(tw) & 1u);
            if (lane == nrows - 1) cut = cut || ((tw >> 61) & 1ull);
            for (int k = 0; k < A.nA; ++k) {
                const double a = __ldcs(g + k * TILE);
                double s = SQUARE ? a * a * yv : a * yv;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const double t = __shfl_up_sync(0xffffffffu, s, d);
                    if (dist >= d) s += t;
                }
                if (tail) {
                    if (!cut) x[ia + k] = fma(cx, x[ia + k], s);
                    else (segStart == 0 ? carryFirst : carryLast)[tile * N_ASTRO + k] = s;
                }
            }
        }
        if (ATT && A.nAtt > 0 && valid) {   // ---- attitude
            const int64_t s = __ldcs(A.iatt + i);
            GSR_ASSERT(s >= 0 && s + 4 <= A.nDof);
            double *xt = x + A.offAtt + s;
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const double v = __ldcs(g + (A.nA + 4 * a + j) * TILE);
                    atomicAdd(xt + a * A.nDof + j, SQUARE ? v * v * yv : v * yv);
                }
        }
        if (valid)   // ---- instrumental
            for (int j = 0; j < A.nI; ++j) {
                const int32_t c = ic_at(A, (tile * A.nI + j) * TILE + lane);
                GSR_ASSERT(c >= 0 && c < A.nInstr);
                const double v = __ldcs(g + (kT + j) * TILE);
                atomicAdd(x + A.offInstr + c, SQUARE ? v * v * yv : v * yv);
            }
        for (int q = 0; q < A.nG; ++q) {   // ---- global columns: fixed-order warp sum into this warp's accumulator
            const double v = __ldcs(g + (kI + q) * TILE);
            const double t = warp_sum(SQUARE ? v * v * yv : v * yv);
            if (lane == 0) gAcc[warp][q] += t;
        }
    }
    __syncthreads();
    if (threadIdx.x < A.nG) {
        double t = 0.0;
        for (int w = 0; w < WARPS; ++w) t += gAcc[w][threadIdx.x];
        globPartial[int64_t(threadIdx.x) * gridDim.x + blockIdx.x] = t;
    }
}

// Astrometric-only layouts (N_Att = N_Instr = N_Glob = 0: the paper's 100 GB dataset "solves the astrometric part",
// PAPER.md:263): the N_Astro <= 5 coefficients of a row are loaded together (predicated on the width, which is uniform over
// the grid) and scanned side by side, instead of one after the other as in k_aprod2_gen (Medium-sized system: 4.1 -> see
// DESIGN.md 5).  Same carries, same fix-up (k_fixup_gen).
template <bool SQUARE>
__global__ void __launch_bounds__(THREADS)
k_aprod2_astro(MatView A, const double *__restrict__ y, double *__restrict__ x, const double *__restrict__ coef,
               double *__restrict__ carryFirst, double *__restrict__ carryLast, const int *done)
{
    if (done && *done) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const double cx = coef[0], cy = coef[1];
    const int64_t nTiles = (A.m + TILE - 1) / TILE;
    const int nA = A.nA;
    for (int64_t tile = int64_t(blockIdx.x) * WARPS + warp; tile < nTiles; tile += int64_t(gridDim.x) * WARPS) {
        const int64_t r0 = tile * TILE;
        const int nrows = int(min(int64_t(TILE), A.m - r0));
        const bool valid = lane < nrows;
        const int ln = valid ? lane : nrows - 1;
        const int64_t i = r0 + ln;
        const double *g = A.V + tile * (int64_t(A.nPar) * TILE) + ln;
        const double yv = valid ? (SQUARE ? 1.0 : cy * y[i]) : 0.0;     // lanes past the last row add zeros
        double s[N_ASTRO];
#pragma unroll
        for (int k = 0; k < N_ASTRO; ++k) {
            const double a = k < nA ? __ldcs(g + k * TILE) : 0.0;
            s[k] = SQUARE ? a * a * yv : a * yv;
        }
        const unsigned long long tw = __ldg(A.tw + tile);
        const int64_t ia = nA * star_of(A, tw, i, ln);
        GSR_ASSERT(ia >= 0 && ia + nA <= A.offAtt);
        const unsigned heads = uint32_t(tw) | 1u;
        if (heads == 1u) {   // one star in the whole tile: totals instead of a scan (see k_aprod2)
            const double tot = warp_sum5(s, lane);
            const int k = (lane >> 2) & 7;
            if ((lane & 3) == 0 && k < nA) {
                if (!(uint32_t(tw) & 1u) || ((tw >> 61) & 1ull)) carryFirst[tile * N_ASTRO + k] = tot;
                else x[ia + k] = fma(cx, x[ia + k], tot);
            }
            continue;
        }
        const bool tail = valid && ((lane == nrows - 1) || ((heads >> 1) >> lane) & 1u);
        const int segStart = 31 - __clz(heads & (0xffffffffu >> (31 - lane)));
        const int dist = lane - segStart;
        bool cut = false;
        if (segStart == 0) cut = !(uint32_t(tw) & 1u);
        if (lane == nrows - 1) cut = cut || ((tw >> 61) & 1ull);
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
#pragma unroll
            for (int k = 0; k < N_ASTRO; ++k) {
                if (k < nA) {   // uniform over the grid
                    const double t = __shfl_up_sync(0xffffffffu, s[k], d);
                    if (dist >= d) s[k] += t;
                }
            }
        }
        if (tail) {
#pragma unroll
            for (int k = 0; k < N_ASTRO; ++k) {
                if (k < nA) {
                    if (!cut) x[ia + k] = fma(cx, x[ia + k], s[k]);
                    else (segStart == 0 ? carryFirst : carryLast)[tile * N_ASTRO + k] = s[k];
                }
            }
        }
    }
}

// Finishes the astro section (stars cut by tile edges, stars without rows) and the global columns of k_aprod2_gen.
__global__ void __launch_bounds__(256)
k_fixup_gen(MatView A, double *__restrict__ x, const double *__restrict__ coef, const double *__restrict__ carryFirst,
            const double *__restrict__ carryLast, const double *__restrict__ globPartial, int nGlobPartial, const int *done)
{
    __shared__ double red[32];
    if (done && *done) return;
    const double cx = coef[0];
    if (blockIdx.x == gridDim.x - 1) {
        for (int q = 0; q < A.nG; ++q) {
            double g = 0.0;
            for (int p = threadIdx.x; p < nGlobPartial; p += blockDim.x) g += globPartial[int64_t(q) * nGlobPartial + p];
            g = block_sum(g, red);
            if (threadIdx.x == 0) x[A.offGlob + q] += g;   // section already scaled by cx
        }
        return;
    }
    const int64_t s = int64_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (s >= A.nStars) return;
    const int64_t r0 = A.rp[s], r1 = A.rp[s + 1];
    double *xa = x + s * A.nA;
    if (r0 == r1) {
        for (int k = 0; k < A.nA; ++k) xa[k] *= cx;
        return;
    }
    const int64_t t0 = r0 / TILE, t1 = (r1 - 1) / TILE;
    if (t0 == t1) return;   // stored by k_aprod2_gen
    for (int k = 0; k < A.nA; ++k) {
        double acc = 0.0;
        for (int64_t t = t0; t <= t1; ++t)
            acc += ((t == t0 && r0 != t * TILE) ? carryLast : carryFirst)[t * N_ASTRO + k];
        xa[k] = fma(cx, xa[k], acc);
    }
}

// ---------------------------------------------------------------------------------------
// Constraint rows ("Constraints kernels"): CSR tail below the
// observation rows.  aprod1: one warp per row; aprod2: one thread per non-zero (RED).
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_con_aprod1(MatView A, const double *__restrict__ x, double *__restrict__ y,
             const double *__restrict__ coef, double *__restrict__ sqPartial, const int *done)
{
    __shared__ double red[32];
    if (done && *done) return;
    const int lane = threadIdx.x & 31;
    const double cx = coef[0], cy = coef[1];
    double sq = 0.0;
    for (int64_t r = (int64_t(blockIdx.x) * blockDim.x + threadIdx.x) >> 5; r < A.nCon;
         r += (int64_t(gridDim.x) * blockDim.x) >> 5) {
        double sum = 0.0;
        for (int64_t q = A.conRp[r] + lane; q < A.conRp[r + 1]; q += 32) {
            GSR_ASSERT(A.conCol[q] >= 0 && A.conCol[q] < A.n);
            sum = fma(A.conVal[q], __ldg(x + A.conCol[q]), sum);
        }
        sum = warp_sum(sum);
        if (lane == 0) {
            const double yi = fma(cy, y[A.m + r], cx * sum);
            y[A.m + r] = yi;
            sq = fma(yi, yi, sq);
        }
    }
    const double b = block_sum(sq, red);
    if (threadIdx.x == 0 && sqPartial) sqPartial[blockIdx.x] = b;
}

template <bool SQUARE>
__global__ void __launch_bounds__(256)
k_con_aprod2(MatView A, const double *__restrict__ y, double *__restrict__ x,
             const double *__restrict__ coef, const int *done)
{
    if (done && *done) return;
    const double cy = coef[1];
    const int lane = threadIdx.x & 31;
    for (int64_t r = (int64_t(blockIdx.x) * blockDim.x + threadIdx.x) >> 5; r < A.nCon;
         r += (int64_t(gridDim.x) * blockDim.x) >> 5) {
        const double yv = SQUARE ? 1.0 : cy * y[A.m + r];
        for (int64_t q = A.conRp[r] + lane; q < A.conRp[r + 1]; q += 32) {
            const double v = A.conVal[q];
            GSR_ASSERT(A.conCol[q] >= 0 && A.conCol[q] < A.n);
            atomicAdd(x + A.conCol[q], SQUARE ? v * v : v * yv);
        }
    }
}

// ---------------------------------------------------------------------------------------
// LSQR vector kernels (not described as ported in the paper).
// ---------------------------------------------------------------------------------------
// partial[b] = sum over this CTA's grid-stride elements of a[j]^2 (Eq. 4 norm, PAPER.md:226,
// in its unscaled form; fixed summation order for a fixed grid).
__global__ void __launch_bounds__(256)
k_sumsq(const double *__restrict__ a, int64_t n, double *__restrict__ partial, const int *done)
{
    __shared__ double red[32];
    if (done && *done) return;
    double s = 0.0;
    for (int64_t j = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; j < n;
         j += int64_t(gridDim.x) * blockDim.x) {
        const double t = a[j];
        s = fma(t, t, s);
    }
    s = block_sum(s, red);
    if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

// Step 4 of LSQR: dk = w/rho; x += t1*w; w = v + t2*w; var += dk^2;
// ddnorm += |dk|^2, with v = v^ * inv_alpha (lazy normalisation of v).
__global__ void __launch_bounds__(256)
k_update(double *__restrict__ x, double *__restrict__ w, const double *__restrict__ vhat,
         double *__restrict__ var, int64_t n, const Scalars *__restrict__ S,
         double *__restrict__ ddPartial)
{
    __shared__ double red[32];
    if (S->done) return;
    const double t1 = S->t1, t2 = S->t2, ir = S->inv_rho, ia = S->inv_alpha;
    double dd = 0.0;
    for (int64_t j = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; j < n;
         j += int64_t(gridDim.x) * blockDim.x) {
        const double wj = w[j];
        const double dk = wj * ir;
        x[j] = fma(t1, wj, x[j]);
        w[j] = fma(t2, wj, vhat[j] * ia);
        var[j] = fma(dk, dk, var[j]);
        dd = fma(dk, dk, dd);
    }
    dd = block_sum(dd, red);
    if (threadIdx.x == 0) ddPartial[blockIdx.x] = dd;
}

// w = v^ * inv_alpha (start of LSQR: w = v)
__global__ void k_init_w(double *__restrict__ w, const double *__restrict__ vhat, int64_t n,
                         const Scalars *__restrict__ S)
{
    const double ia = S->inv_alpha;
    for (int64_t j = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; j < n;
         j += int64_t(gridDim.x) * blockDim.x)
        w[j] = vhat[j] * ia;
}

// gsr_set_cov_pairs: first couple with an index outside [0, n)
__global__ void k_validate_pairs(const int64_t *__restrict__ pi, const int64_t *__restrict__ pj, int64_t npairs, int64_t n,
                                 unsigned long long *bad)
{
    for (int64_t q = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; q < npairs; q += int64_t(gridDim.x) * blockDim.x)
        if (pi[q] < 0 || pi[q] >= n || pj[q] < 0 || pj[q] >= n) atomicMin(bad, (unsigned long long)q);
}

// Covariances of the caller's couples of unknowns (Alg. 1 l.26; R26), accumulated
// beside the variances: acc[q] += d_k[i] d_k[j] with d_k = w_k / rho_k.  Runs BEFORE k_update of the same iteration (which
// overwrites w), after the scalar kernel that set inv_rho.  One thread per couple; couples are few (<< n).
__global__ void k_cov_update(const double *__restrict__ w, const int64_t *__restrict__ pi, const int64_t *__restrict__ pj,
                             int64_t npairs, const Scalars *__restrict__ S, double *__restrict__ acc)
{
    if (S->done) return;
    const double ir = S->inv_rho;
    for (int64_t q = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; q < npairs; q += int64_t(gridDim.x) * blockDim.x)
        acc[q] = fma(w[pi[q]] * ir, w[pj[q]] * ir, acc[q]);
}

// Alg. 1 l.27 for the couples: cov(i, j) = p_i p_j s^2 acc, s as in k_finish, so that cov(i, i) = se_i^2.
__global__ void k_cov_finish(const double *__restrict__ acc, const int64_t *__restrict__ pi, const int64_t *__restrict__ pj,
                             int64_t npairs, const double *__restrict__ p, int64_t n, int64_t mTot,
                             const Scalars *__restrict__ S, double *__restrict__ out)
{
    double s = S->rnorm;
    if (mTot > n) s = s / sqrt(double(mTot - n));
    for (int64_t q = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; q < npairs; q += int64_t(gridDim.x) * blockDim.x)
        out[q] = p[pi[q]] * p[pj[q]] * (acc[q] * (s * s));
}

// Alg. 1 l.27: x = p (.) z, se = p (.) sqrt(var) * rnorm / sqrt(m - n).
__global__ void k_finish(const double *__restrict__ z, const double *__restrict__ var,
                         const double *__restrict__ p, double *__restrict__ xOut,
                         double *__restrict__ seOut, int64_t n, int64_t mTot,
                         const Scalars *__restrict__ S)
{
    double s = S->rnorm;
    if (mTot > n) s = s / sqrt(double(mTot - n));
    for (int64_t j = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; j < n;
         j += int64_t(gridDim.x) * blockDim.x) {
        xOut[j] = p[j] * z[j];
        if (seOut) seOut[j] = p[j] * (sqrt(var[j]) * s);
    }
}

// ---------------------------------------------------------------------------------------
// Scalar recurrences and stop tests (Paige & Saunders 1982, cited
// PAPER.md:34, 742-743), one CTA; the partial sums are reduced in a fixed order first.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ double reduce_partials(const double *p, int n, double *red)
{
    double s = 0.0;
    for (int j = threadIdx.x; j < n; j += blockDim.x) s += p[j];
    s = block_sum(s, red);
    __shared__ double bc;
    if (threadIdx.x == 0) bc = s;
    __syncthreads();
    return bc;
}

enum { PH_INIT_BETA = 0, PH_INIT_ALPHA = 1, PH_AFTER_APROD1 = 2, PH_AFTER_APROD2 = 3, PH_AFTER_UPDATE = 4 };

__global__ void __launch_bounds__(256)
k_scalar(int phase, Scalars *S, const double *partial, int nPartial, double *trace, int traceCap)
{
    __shared__ double red[32];
    if (phase >= PH_AFTER_APROD1 && S->done) return;
    const double sum = reduce_partials(partial, nPartial, red);
    if (threadIdx.x != 0) return;
    if (phase == PH_INIT_BETA) {
        // step 1: beta = |b|, u = b/beta (lazy: u^ = b, scale kept in beta)
        const double beta = sqrt(sum);
        S->beta = beta; S->bnorm = beta; S->rnorm = beta; S->phibar = beta;
        S->a2_cx = 1.0; S->a2_cy = beta > 0.0 ? 1.0 / beta : 0.0;
        S->anorm = 0; S->acond = 0; S->ddnorm = 0; S->xxnorm = 0; S->xnorm = 0; S->z = 0;
        S->cs2 = -1.0; S->sn2 = 0.0; S->arnorm = 0; S->itn = 0; S->istop = 0; S->done = 0;
        S->alpha = 0;
    } else if (phase == PH_INIT_ALPHA) {
        // v = A^T u, alpha = |v|, v /= alpha (lazy), w = v
        const double alpha = sqrt(sum);
        S->alpha = alpha; S->rhobar = alpha;
        S->inv_alpha = alpha > 0.0 ? 1.0 / alpha : 0.0;
        S->arnorm = alpha * S->beta;
        if (S->arnorm == 0.0) S->done = 1;         // x = 0 is the solution: istop 0, itn 0
        if (S->itnlim <= 0) S->done = 1;
        S->a1_cx = S->inv_alpha;
        S->a1_cy = S->beta > 0.0 ? -alpha / S->beta : 0.0;
    } else if (phase == PH_AFTER_APROD1) {
        // step 2 first half: beta = |A v - alpha u|, anorm; coefficients of v <- A^T u - beta v
        const double beta = sqrt(sum), alpha = S->alpha;
        S->beta = beta;
        if (beta > 0.0) {
            S->anorm = sqrt(S->anorm * S->anorm + alpha * alpha + beta * beta);
            S->a2_cy = 1.0 / beta;
            S->a2_cx = -beta * S->inv_alpha;       // v = v^/alpha
        } else {
            S->a2_cy = 0.0; S->a2_cx = 1.0;
        }
    } else if (phase == PH_AFTER_APROD2) {
        // step 2 second half + step 3 (plane rotation) + coefficients of step 4
        const double beta = S->beta;
        double alpha = sqrt(sum);
        if (!(beta > 0.0)) alpha = S->alpha;       // aprod2 was skipped: v, alpha unchanged
        S->alpha = alpha;
        S->inv_alpha = alpha > 0.0 ? 1.0 / alpha : 0.0;
        const double rhobar = S->rhobar, phibar = S->phibar;
        const double rho = sqrt(rhobar * rhobar + beta * beta);
        const double cs = rhobar / rho, sn = beta / rho;
        const double theta = sn * alpha;
        S->rhobar = -cs * alpha;
        const double phi = cs * phibar;
        S->phibar = sn * phibar;
        const double tau = sn * phi;
        S->t1 = phi / rho; S->t2 = -theta / rho; S->inv_rho = 1.0 / rho;
        // step 5: norm of x
        const double delta = S->sn2 * rho, gambar = -S->cs2 * rho;
        const double rhs = phi - delta * S->z;
        const double zbar = rhs / gambar;
        S->xnorm = sqrt(S->xxnorm + zbar * zbar);
        const double gamma = sqrt(gambar * gambar + theta * theta);
        S->cs2 = gambar / gamma; S->sn2 = theta / gamma;
        S->z = rhs / gamma;
        S->xxnorm = S->xxnorm + S->z * S->z;
        S->rnorm = S->phibar;
        S->arnorm = alpha * fabs(tau);
    } else {  // PH_AFTER_UPDATE: steps 6-7
        S->ddnorm = S->ddnorm + sum;
        S->itn = S->itn + 1;
        const double anorm = S->anorm, rnorm = S->rnorm, arnorm = S->arnorm, xnorm = S->xnorm;
        const double bnorm = S->bnorm;
        S->acond = anorm * sqrt(S->ddnorm);
        if (trace) {
            double *t = trace + 5 * ((S->itn - 1) % traceCap);
            t[0] = rnorm; t[1] = arnorm; t[2] = anorm; t[3] = S->acond; t[4] = xnorm;
        }
        const double test1 = rnorm / bnorm;
        const double test2 = (anorm * rnorm != 0.0) ? arnorm / (anorm * rnorm) : 0.0;
        const double test3 = 1.0 / S->acond;
        const double t1p = test1 / (1.0 + anorm * xnorm / bnorm);
        const double rtol = S->btol + S->atol * anorm * xnorm / bnorm;
        int istop = 0;
        if (S->itn >= S->itnlim) istop = 7;
        if (1.0 + test3 <= 1.0) istop = 6;
        if (1.0 + test2 <= 1.0) istop = 5;
        if (1.0 + t1p <= 1.0) istop = 4;
        if (test3 <= S->ctol) istop = 3;
        if (test2 <= S->atol) istop = 2;
        if (test1 <= rtol) istop = 1;
        S->istop = istop;
        if (istop) S->done = 1;
        // coefficients of the next aprod1:  u^ <- (1/alpha) A v^ - (alpha/beta) u^
        S->a1_cx = S->inv_alpha;
        S->a1_cy = S->beta > 0.0 ? -S->alpha / S->beta : 0.0;
    }
}

// ---------------------------------------------------------------------------------------
// Setup kernels: validation, star row pointer, preconditioner.
// ---------------------------------------------------------------------------------------
__global__ void k_validate(MatView A, unsigned long long *badRow)
{
    for (int64_t i = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; i < A.m;
         i += int64_t(gridDim.x) * blockDim.x) {
        // k_ingest_index stored -1 for a matrixIndexAstro that is not 5*star with star in [0, nStars) and for a
        // matrixIndexAtt outside [0, nDof-4]; k_ingest_rows stored -1 in star[] for a row with a column that does not
        // fit 2 bytes (star[] is the per-row mark of the upload for every layout: zeros when there is no astro section)
        bool bad = A.star[i] < 0 || (A.nAtt > 0 && A.iatt[i] < 0);
        if (A.nA > 0 && i > 0) bad = bad || A.star[i - 1] > A.star[i];
        for (int j = 0; j < A.nI; ++j) {
            const int32_t c = ic_at(A, cpos(i, j, A.nI));
            bad = bad || c < 0 || c >= A.nInstr;
        }
        if (bad) atomicMin(badRow, (unsigned long long)i);
    }
}

// rp[s] = first row i with star[i] >= s  (rows sorted by star), s = 0..nStars
__global__ void k_star_rowptr(const int32_t *__restrict__ star, int64_t m, int64_t nStars,
                              int64_t *__restrict__ rp)
{
    const int64_t s = int64_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (s > nStars) return;
    int64_t lo = 0, hi = m;
    while (lo < hi) {
        const int64_t mid = (lo + hi) >> 1;
        if (star[mid] < s) lo = mid + 1; else hi = mid;
    }
    rp[s] = lo;
}

// tw[tile] from the validated per-row star array (see MatView::tw)
__global__ void k_tile_words(const int32_t *__restrict__ star, int64_t m, unsigned long long *__restrict__ tw)
{
    const int lane = threadIdx.x & 31;
    const int64_t nTiles = (m + TILE - 1) / TILE;
    for (int64_t tile = (int64_t(blockIdx.x) * blockDim.x + threadIdx.x) >> 5; tile < nTiles;
         tile += (int64_t(gridDim.x) * blockDim.x) >> 5) {
        const int64_t r0 = tile * TILE;
        const int nrows = int(min(int64_t(TILE), m - r0));
        const int64_t i = r0 + min(lane, nrows - 1);
        const int32_t s = star[i];
        const int32_t sp = i > 0 ? star[i - 1] : -1;
        const bool head = lane < nrows && s != sp;
        const bool gap = lane < nrows && lane > 0 && s > sp + 1;
        const unsigned hm = __ballot_sync(0xffffffffu, head);
        const unsigned gm = __ballot_sync(0xffffffffu, gap);
        if (lane == 0) {
            const int64_t last = r0 + nrows - 1;
            const bool contNext = last + 1 < m && star[last + 1] == star[last];
            tw[tile] = (unsigned long long)hm | ((unsigned long long)uint32_t(s) << 32) | (contNext ? 1ull << 61 : 0ull) |
                       (gm ? 1ull << 62 : 0ull);
        }
    }
}

// Upload: matrixIndexAstro / matrixIndexAtt (i64, "M_i") -> 4-byte star and attitude start;
// a value that breaks its contract becomes -1 and is reported by k_validate.
// nA: astrometric unknowns per star (matrixIndexAstro = nA*star); a section that is absent passes a null array.
__global__ void k_ingest_index(int64_t cnt, const int64_t *__restrict__ ia, const int64_t *__restrict__ iatt,
                               int64_t nStars, int64_t nDof, int nA, int32_t *__restrict__ star, int32_t *__restrict__ att)
{
    for (int64_t q = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; q < cnt;
         q += int64_t(gridDim.x) * blockDim.x) {
        if (ia) {
            const int64_t a = ia[q];
            star[q] = (a >= 0 && a % nA == 0 && a / nA < nStars) ? int32_t(a / nA) : -1;
        }
        if (iatt) {
            const int64_t s = iatt[q];
            att[q] = (s >= 0 && s <= nDof - 4) ? int32_t(s) : -1;
        }
    }
}

__global__ void k_validate_con(MatView A, int64_t nnz, unsigned long long *badRow)
{
    for (int64_t q = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; q < nnz;
         q += int64_t(gridDim.x) * blockDim.x) {
        const int64_t c = A.conCol[q];
        if (c < 0 || c >= A.n) atomicMin(badRow, (unsigned long long)q);
    }
    for (int64_t r = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; r <= A.nCon;
         r += int64_t(gridDim.x) * blockDim.x) {
        const int64_t a = A.conRp[r];
        bool bad = a < 0 || a > nnz || (r == 0 && a != 0) || (r == A.nCon && a != nnz);
        if (r > 0) bad = bad || A.conRp[r - 1] > a;
        if (bad) atomicMin(badRow, (unsigned long long)r);
    }
}

// p_j = 1/sqrt(colsq_j), or 1 for an empty column (readings R1-R2)
__global__ void k_colscale(double *__restrict__ p, int64_t n)
{
    for (int64_t j = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; j < n;
         j += int64_t(gridDim.x) * blockDim.x) {
        const double s = p[j];
        p[j] = s > 0.0 ? 1.0 / sqrt(s) : 1.0;
    }
}

// A_ij <- fl(A_ij * p_j) in place ("Normalization of A by p", Alg. 1 l.3).
// One thread per stored coefficient (coalesced over A_d).
__global__ void k_scale_values(MatView A, const double *__restrict__ p)
{
    const int64_t total = ((A.m + TILE - 1) / TILE) * (int64_t(A.nPar) * TILE);
    const int kT = A.nA + A.nAtt, kI = kT + A.nI;
    for (int64_t e = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; e < total;
         e += int64_t(gridDim.x) * blockDim.x) {
        // e = (tile*nPar + k)*32 + lane
        const int64_t tk = e >> 5;
        const int64_t tile = tk / A.nPar;
        const int k = int(tk - tile * A.nPar);
        const int64_t i = tile * TILE + (e & 31);
        if (i >= A.m) continue;
        int64_t c;
        if (k < A.nA) c = A.nA * star_of(A, A.tw[tile], i, int(e & 31)) + k;
        else if (k < kT) c = A.offAtt + ((k - A.nA) >> 2) * A.nDof + A.iatt[i] + ((k - A.nA) & 3);
        else if (k < kI) c = A.offInstr + ic_at(A, cpos(i, k - kT, A.nI));
        else c = A.offGlob + (k - kI);
        A.V[e] = A.V[e] * p[c];
    }
}

__global__ void k_scale_con_values(MatView A, int64_t nnz, const double *__restrict__ p)
{
    for (int64_t q = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; q < nnz;
         q += int64_t(gridDim.x) * blockDim.x)
        A.conVal[q] = A.conVal[q] * p[A.conCol[q]];
}

// Upload (Alg. 1 l.6-12): rows [row0, row0+cnt) arrive row-major (A_d, I_c as the paper
// stores them) and are written tile-transposed.  One thread per stored element; the
// reads are coalesced, the writes hit 32 lines per warp but only once per upload.
// A column outside [0, nInstr) cannot be stored in 2 bytes: it is written as column 0 and the row is marked bad in the
// upload scratch (rowMark[i] = -1, the value k_ingest_index gives a broken star index), where k_validate finds it.  The mark
// lives with the row: sending the row again rewrites it, so an abandoned upload leaves nothing behind.
__global__ void k_ingest_rows(MatView A, int32_t *__restrict__ icDev, uint16_t *__restrict__ ic16Dev, int64_t row0, int64_t cnt,
                              const double *__restrict__ values, const int32_t *__restrict__ ic,
                              int32_t *rowMark)
{
    const int64_t nV = cnt * A.nPar, nC = cnt * A.nI;
    for (int64_t e = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; e < nV + nC;
         e += int64_t(gridDim.x) * blockDim.x) {
        if (e < nV) {
            const int64_t r = e / A.nPar;
            A.V[vpos(row0 + r, int(e - r * A.nPar), A.nPar)] = values[e];
        } else {
            const int64_t f = e - nV, r = f / A.nI;
            const int32_t c = ic[f];
            if (ic16Dev) {
                const bool ok = c >= 0 && c < A.nInstr;
                ic16Dev[cpos(row0 + r, int(f - r * A.nI), A.nI)] = ok ? uint16_t(c) : uint16_t(0);
                if (!ok) rowMark[row0 + r] = -1;
            } else {
                icDev[cpos(row0 + r, int(f - r * A.nI), A.nI)] = c;
            }
        }
    }
}

// out[(i - row0)*nPar + k] = V(i, k) for rows [row0, row0+cnt): the row-major view for gsr_get_values.
__global__ void k_export_rows(MatView A, int64_t row0, int64_t cnt, double *__restrict__ out)
{
    const int64_t nV = cnt * A.nPar;
    for (int64_t e = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; e < nV;
         e += int64_t(gridDim.x) * blockDim.x) {
        const int64_t r = e / A.nPar;
        out[e] = A.V[vpos(row0 + r, int(e - r * A.nPar), A.nPar)];
    }
}

// Setup: how uneven is the use of the instrument columns?  cnt[c] = number of coefficients in column c;
// the largest count against the mean decides whether aprod2 pre-sums equal columns inside a warp.
__global__ void k_instr_hist(MatView A, unsigned int *__restrict__ cnt)
{
    const int64_t total = ((A.m + TILE - 1) / TILE) * (int64_t(A.nI) * TILE);
    for (int64_t e = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; e < total;
         e += int64_t(gridDim.x) * blockDim.x) {
        const int64_t i = (e / (A.nI * TILE)) * TILE + (e & 31);
        if (i < A.m) atomicAdd(cnt + ic_at(A, e), 1u);
    }
}
__global__ void k_max_u32(const unsigned int *__restrict__ cnt, int64_t n, unsigned int *__restrict__ out)
{
    unsigned int mx = 0;
    for (int64_t j = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; j < n; j += int64_t(gridDim.x) * blockDim.x)
        mx = max(mx, cnt[j]);
    mx = __reduce_max_sync(0xffffffffu, mx);
    if ((threadIdx.x & 31) == 0) atomicMax(out, mx);
}

__global__ void k_fill(double *__restrict__ a, int64_t n, double v)
{
    for (int64_t j = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; j < n;
         j += int64_t(gridDim.x) * blockDim.x)
        a[j] = v;
}

}  // namespace gsr
