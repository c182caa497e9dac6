// bie_gemv.cuh -- SURVEY 8(a) row a6: the dense FP64 GEMV y = A x of the Krylov matvec (PAPER.md:L857,
// "level 2 BLAS speed" PAPER.md:L921), as a CTA-level device function shared by bie_matvec and by the
// persistent GMRES kernel.  HBM-bound: 8 B read per entry, 2 flops.
//
// A CTA owns a contiguous block of rows [r0, r1).  Work is cut into units of (row pair) x (column chunk
// of gemv_chunk() doubles); the CTA's warps take units round-robin, so every warp has the same number of
// 128-bit loads to issue however the rows divide.  A warp streams its two rows with 2 x GEMV_UNROLL
// independent LDG.128 per lane in flight (512 contiguous bytes per warp-load), multiplies by x from shared
// memory (or from L2 when n is too large for shared memory), reduces by warp shuffles and leaves the
// partial sum in shared memory; partials are then summed over chunks in fixed order (deterministic).
#pragma once
#include "bie_common.cuh"

#define GEMV_UNROLL 4

// doubles per (row, chunk) unit: 2048 (32 warp-loads of 64 doubles) for large n; smaller for small n so
// that every warp of the CTA still gets a unit.  Always a multiple of 64.
__host__ __device__ inline int gemv_chunk(int rows_per_cta, int n, int nwarp)
{
    int chunk = 2048;
    const int npair = (rows_per_cta + 1) >> 1;
    while (chunk > 128 && npair * ((n + chunk - 1) / chunk) < 2 * nwarp) chunk >>= 1;
    // equal chunks: a short last chunk would always land on the same warps (units go round-robin)
    const int nch = (n + chunk - 1) / chunk;
    chunk = ((n + nch - 1) / nch + 63) & ~63;
    return chunk;
}

// streaming (evict-first) 128-bit load for matrices larger than L2; plain read-only load otherwise
template <bool STREAM>
__device__ __forceinline__ double2 gemv_ld(const double2* p)
{
    if (STREAM) return __ldcs(p);
    return __ldg(p);
}

// number of doubles of shared memory bie_cta_gemv needs for partial sums
__host__ __device__ inline int gemv_part_doubles(int rows_per_cta, int n, int chunk)
{
    const int nch = (n + chunk - 1) / chunk;
    return nch * ((rows_per_cta + 1) & ~1);
}

// y_local[r - r0] = sum_c A[r][c] * x[c] for r in [r0, r1).  xs: x in shared memory (XS = true) or global.
// part: shared scratch of gemv_part_doubles() doubles.  All threads of the team must call; ends with the
// results in y_local (shared) after a team barrier.  n = number of columns used (the hybrid operator passes
// the width of its stored slab).
// 128-bit load with an L2 eviction-priority hint (policy from createpolicy): the resident part of a streamed matrix
__device__ __forceinline__ double2 gemv_ld_hint(const double2* p, unsigned long long pol)
{
    double2 v;
    asm volatile("ld.global.nc.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol));
    return v;
}

// one (row pair) x (column chunk) unit of a warp: acc0/acc1 += A[ra..ra+1][cbeg..cend) . x
// STR: 0 default policy (__ldg), 1 streaming (evict-first), 2 keep (L2 evict-last hint `pol`)
template <int STR, bool XS, int UNROLL>
__device__ __forceinline__ void gemv_unit(const double2* __restrict__ a0, const double2* __restrict__ a1, int cbeg, int cend,
                                          int lane, const double* xs, double& acc0, double& acc1, unsigned long long pol = 0)
{
    auto ld = [&](const double2* q) { return STR == 2 ? gemv_ld_hint(q, pol) : (STR == 1 ? __ldcs(q) : __ldg(q)); };
    int c = cbeg + lane;
    for (; c + 32 * (UNROLL - 1) < cend; c += 32 * UNROLL) {
        double2 v0[UNROLL], v1[UNROLL];
#pragma unroll
        for (int i = 0; i < UNROLL; ++i) {
            v0[i] = ld(a0 + c + 32 * i);
            v1[i] = ld(a1 + c + 32 * i);
        }
#pragma unroll
        for (int i = 0; i < UNROLL; ++i) {
            double2 xv;
            if (XS) xv = reinterpret_cast<const double2*>(xs)[c + 32 * i];
            else xv = __ldcg(reinterpret_cast<const double2*>(xs) + c + 32 * i);
            acc0 = fma(v0[i].x, xv.x, acc0); acc0 = fma(v0[i].y, xv.y, acc0);
            acc1 = fma(v1[i].x, xv.x, acc1); acc1 = fma(v1[i].y, xv.y, acc1);
        }
    }
    for (; c < cend; c += 32) {
        const double2 v0 = ld(a0 + c), v1 = ld(a1 + c);
        double2 xv;
        if (XS) xv = reinterpret_cast<const double2*>(xs)[c];
        else xv = __ldcg(reinterpret_cast<const double2*>(xs) + c);
        acc0 = fma(v0.x, xv.x, acc0); acc0 = fma(v0.y, xv.y, acc0);
        acc1 = fma(v1.x, xv.x, acc1); acc1 = fma(v1.y, xv.y, acc1);
    }
}

// res_pairs (STREAM only): the first res_pairs row pairs of the CTA's block are read with the default cache policy and stay
// in the 126 MB L2 from one application to the next; the others are streamed (evict-first) so that they do not displace
// them.  For a matrix a little larger than L2 (n = 3500 ... 7000) this removes most of the HBM traffic of a GEMV.
template <bool STREAM, bool XS, int UNROLL = GEMV_UNROLL>
__device__ __forceinline__ void bie_cta_gemv(const double* __restrict__ A, long long lda, int n, int r0, int r1, int chunk,
                                             const double* xs, double* part, double* y_local, const Team& tm,
                                             int res_pairs = 0)
{
    const int lane = tm.tid & 31, warp = tm.warp, nwarp = tm.nwarp;
    const int rows = r1 - r0;
    const int rows2 = (rows + 1) & ~1;
    const int npair = rows2 >> 1;
    const int nch = (n + chunk - 1) / chunk;
    const int nunit = npair * nch;
    const int n2 = n >> 1;  // double2 columns (lda even: every row is 16-byte aligned)
    unsigned long long keep = 0;
    if (STREAM && res_pairs > 0) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(keep));
    for (int u = warp; u < nunit; u += nwarp) {
        // consecutive warps take consecutive chunks of the same row pair
        const int p = u / nch, ch = u - p * nch;
        const int ra = r0 + 2 * p;
        const bool two = (ra + 1 < r1);
        const double2* a0 = reinterpret_cast<const double2*>(A + (long long)ra * lda);
        const double2* a1 = reinterpret_cast<const double2*>(A + (long long)(two ? ra + 1 : ra) * lda);
        const int cbeg = ch * (chunk >> 1);
        const int cend = min(cbeg + (chunk >> 1), n2);
        double acc0 = 0.0, acc1 = 0.0;
        if (STREAM && p >= res_pairs) gemv_unit<1, XS, UNROLL>(a0, a1, cbeg, cend, lane, xs, acc0, acc1);
        else if (STREAM) gemv_unit<2, XS, UNROLL>(a0, a1, cbeg, cend, lane, xs, acc0, acc1, keep);
        else gemv_unit<0, XS, UNROLL>(a0, a1, cbeg, cend, lane, xs, acc0, acc1);
        if ((n & 1) && ch == nch - 1 && lane == 0) {  // odd n: the last column
            const double xl = XS ? xs[n - 1] : __ldcg(xs + n - 1);
            acc0 = fma(A[(long long)ra * lda + n - 1], xl, acc0);
            if (two) acc1 = fma(A[(long long)(ra + 1) * lda + n - 1], xl, acc1);
        }
        acc0 = bie_warp_sum(acc0);
        acc1 = bie_warp_sum(acc1);
        if (lane == 0) {
            part[ch * rows2 + 2 * p] = acc0;
            part[ch * rows2 + 2 * p + 1] = acc1;
        }
    }
    team_sync(tm);
    for (int r = tm.tid; r < rows; r += tm.nthr) {
        double s = 0.0;
        for (int ch = 0; ch < nch; ++ch) s += part[ch * rows2 + r];
        y_local[r] = s;
    }
    team_sync(tm);
}

// ---------------------------------------------------------------------------------------------------
// Block ring of the hybrid operator (bie_gmres.cu): the stored leading block A[0:nd, 0:nd) arrives in shared memory
// by bulk copies (cp.async.bulk, the TMA engine) issued by ONE thread, as tiles of RING_ROWS rows x one column chunk
// TOGETHER with the chunk of x they multiply, into a ring of RING_STAGES buffers guarded by mbarriers.  No warp has
// to keep loads in flight: the warps that run the pair loops of the recomputed part consume landed tiles between
// their source chunks (they own the issue slots; a tile costs about 150 instructions), claim them through a shared
// counter and leave the tile's row sums in `part`, one slot per (chunk, row): the result does not depend on which
// warp took which tile.  Every CTA streams an equal share of the block's rows, whoever owns them in the solve.
// ---------------------------------------------------------------------------------------------------
#ifndef RING_STAGES
#define RING_STAGES 4
#endif
#define RING_ROWS BIE_TILE_ROWS      // a ring tile is a tile of the block format (bie_common.cuh): ONE 16 KB bulk copy

// doubles per (row, chunk) of a ring tile = BIE_TILE_COLS
__host__ __device__ inline int ring_chunk(int /*rows_per_cta*/, int /*nd*/, int /*nwarp*/) { return BIE_TILE_COLS; }
// shared memory of the ring: RING_STAGES tiles of (RING_ROWS + 1) x chunk doubles, then 2 RING_STAGES mbarriers and the
// tile counter (padded to an even number of doubles)
__host__ __device__ inline int ring_doubles(int chunk) { return RING_STAGES * (RING_ROWS + 1) * chunk + 2 * RING_STAGES + 2; }
// row sums of the tiles: [chunks][rows rounded up to RING_ROWS]
__host__ __device__ inline int ring_part_doubles(int rows_per_cta, int nd, int chunk)
{
    return ((nd + chunk - 1) / chunk) * (((rows_per_cta + RING_ROWS - 1) / RING_ROWS) * RING_ROWS);
}

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_test(unsigned bar, unsigned parity)
{
    unsigned ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
// non-blocking probe (try_wait may suspend the thread for a hardware-defined time before it answers "not yet")
__device__ __forceinline__ bool mbar_probe(unsigned bar, unsigned parity)
{
    unsigned ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    while (!mbar_test(bar, parity)) { }
}
// bulk copy global -> shared of `bytes` (multiple of 16; both addresses 16-byte aligned), completion on `bar`
template <bool HINT>
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned bar, unsigned long long pol)
{
    if (HINT)
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                     :: "r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(pol) : "memory");
    else
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     :: "r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

struct BlockRing {
    const double* A;          // stored block in the block format (bie_common.cuh)
    int nd, r0, r1, chunk;    // columns (= rows) of the block, the rows this CTA streams, doubles per (row, chunk)
    int nch, nunit;           // chunks per row, tiles of one application
    unsigned full0, empty0;   // shared addresses of the mbarriers: full[s] = full0 + 8 s, empty[s] = empty0 + 8 s
    int* next;                // shared: next tile to claim; next[1] = tiles the producer has issued in this application
    const double* stage;      // shared: RING_STAGES tiles of (RING_ROWS + 1) x chunk doubles (rows, then x)
    double* part;             // shared: [nch][rowsP] row sums of the tiles
    int rowsP;
    unsigned long long tile0; // tiles issued before this application (ring position and phase run on across applications)
};

// all threads of the CTA, once per kernel
__device__ __forceinline__ void ring_init(double* ring_mem, int chunk)
{
    if (threadIdx.x == 0) {
        const unsigned b = smem_u32(ring_mem + RING_STAGES * (RING_ROWS + 1) * chunk);
        for (int s = 0; s < 2 * RING_STAGES; ++s) mbar_init(b + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
}

// ONE thread: every tile of the application, in unit order, as ring slots become free
template <bool STREAM>
__device__ __forceinline__ void ring_produce(const BlockRing& R, const double* xin)
{
    unsigned long long pol = 0;
    if (STREAM) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    const unsigned stage_addr = smem_u32(R.stage);
    for (int t = 0; t < R.nunit; ++t) {
        const unsigned long long gidx = R.tile0 + t;
        const unsigned s = (unsigned)(gidx % RING_STAGES), use = (unsigned)(gidx / RING_STAGES);
        mbar_wait(R.empty0 + 8 * s, (use & 1u) ^ 1u);
        const int p = t / R.nch, ch = t - p * R.nch;
        const int cbeg = ch * R.chunk, cend = min(cbeg + R.chunk, R.nd);
        const unsigned xbytes = 8u * (unsigned)(cend - cbeg);
        const unsigned tbytes = 8u * RING_ROWS * BIE_TILE_COLS;
        const unsigned dst = stage_addr + s * (unsigned)(8 * (RING_ROWS + 1) * R.chunk);
        mbar_arrive_expect_tx(R.full0 + 8 * s, tbytes + xbytes);
        bulk_g2s<STREAM>(dst, R.A + ((long long)(R.r0 / RING_ROWS + p) * R.nch + ch) * (RING_ROWS * BIE_TILE_COLS), tbytes,
                         R.full0 + 8 * s, pol);
        bulk_g2s<false>(dst + tbytes, xin + cbeg, xbytes, R.full0 + 8 * s, 0);   // x: L2-resident
        // a consumer may wait for tile t only from here on: mbarrier waits tell phases apart by parity alone, and the
        // previous use of this slot has completed now
        *reinterpret_cast<volatile int*>(R.next + 1) = t + 1;
    }
}

// a whole warp: multiplies tile t (claimed by this warp) with its x chunk as soon as it has landed
__device__ __forceinline__ void ring_tile(const BlockRing& R, int t)
{
    const int lane = threadIdx.x & 31;
    const unsigned long long gidx = R.tile0 + t;
    const unsigned s = (unsigned)(gidx % RING_STAGES), use = (unsigned)(gidx / RING_STAGES);
    const int p = t / R.nch, ch = t - p * R.nch;
    const int nr = min(RING_ROWS, R.r1 - (R.r0 + RING_ROWS * p));
    const int cbeg = ch * R.chunk, cend = min(cbeg + R.chunk, R.nd);
    const int n2 = (cend - cbeg) >> 1;
    while (*reinterpret_cast<volatile int*>(R.next + 1) <= t) { }     // issued (see ring_produce)
    mbar_wait(R.full0 + 8 * s, use & 1u);
    const double2* a = reinterpret_cast<const double2*>(R.stage + (size_t)s * (RING_ROWS + 1) * R.chunk);
    const int ch2 = R.chunk >> 1;
    const double2* x2 = a + RING_ROWS * ch2;
    double acc[RING_ROWS], bcc[RING_ROWS];
#pragma unroll
    for (int i = 0; i < RING_ROWS; ++i) { acc[i] = 0.0; bcc[i] = 0.0; }
    // rows the tile does not have are read anyway (stale shared memory, finite or not) and their sums dropped
    int c = lane;
    if (RING_ROWS <= 4) {
        for (; c + 32 < n2; c += 64) {
            const double2 xa = x2[c], xb = x2[c + 32];
            double2 va[RING_ROWS], vb[RING_ROWS];
#pragma unroll
            for (int i = 0; i < RING_ROWS; ++i) { va[i] = a[i * ch2 + c]; vb[i] = a[i * ch2 + c + 32]; }
#pragma unroll
            for (int i = 0; i < RING_ROWS; ++i) {
                acc[i] = fma(va[i].x, xa.x, acc[i]); bcc[i] = fma(va[i].y, xa.y, bcc[i]);
                acc[i] = fma(vb[i].x, xb.x, acc[i]); bcc[i] = fma(vb[i].y, xb.y, bcc[i]);
            }
        }
    }
    for (; c < n2; c += 32) {
        const double2 xa = x2[c];
        double2 va[RING_ROWS];
#pragma unroll
        for (int i = 0; i < RING_ROWS; ++i) va[i] = a[i * ch2 + c];
#pragma unroll
        for (int i = 0; i < RING_ROWS; ++i) { acc[i] = fma(va[i].x, xa.x, acc[i]); bcc[i] = fma(va[i].y, xa.y, bcc[i]); }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(R.empty0 + 8 * s);     // the slot may be refilled
#pragma unroll
    for (int i = 0; i < RING_ROWS; ++i) {
        const double v = bie_warp_sum(acc[i] + bcc[i]);
        if (lane == 0 && i < nr) R.part[ch * R.rowsP + RING_ROWS * p + i] = v;
    }
}

// a whole warp: claims the next tile and multiplies it; returns false when none is left.  Blocks until the tile has landed.
__device__ __forceinline__ bool ring_consume(const BlockRing& R)
{
    int t = 0;
    if ((threadIdx.x & 31) == 0) t = atomicAdd(R.next, 1);
    t = __shfl_sync(0xffffffffu, t, 0);
    if (t >= R.nunit) return false;
    ring_tile(R, t);
    return true;
}

// a whole warp: the next unclaimed tile if it has ALREADY landed and this warp wins the claim, else -1 (never blocks:
// two shared-memory reads, one mbarrier probe, one compare-and-swap)
__device__ __forceinline__ int ring_try_claim(const BlockRing& R)
{
    const int t = *reinterpret_cast<volatile int*>(R.next);
    if (t >= R.nunit || *reinterpret_cast<volatile int*>(R.next + 1) <= t) return -1;
    const unsigned long long gidx = R.tile0 + t;
    if (!mbar_probe(R.full0 + 8 * (unsigned)(gidx % RING_STAGES), (unsigned)(gidx / RING_STAGES) & 1u)) return -1;
    int won = 0;
    if ((threadIdx.x & 31) == 0) won = (atomicCAS(R.next, t, t + 1) == t);
    won = __shfl_sync(0xffffffffu, won, 0);
    return won ? t : -1;
}
// not inlined: the pair loops around the call keep their register allocation
static __device__ __noinline__ void ring_tile_call(const BlockRing& R, int t) { ring_tile(R, t); }

// what the pair loops of bie_free.cuh call between source chunks
struct NoPoll { __device__ __forceinline__ void operator()() const {} };
struct RingPoll {
    const BlockRing* R;
    int max_tiles;
    // a whole warp, between two source chunks of its pair loop: takes up to max_tiles tiles that have ALREADY landed
    __device__ __forceinline__ void operator()() const
    {
        for (int k = 0; k < max_tiles; ++k) {
            const int t = ring_try_claim(*R);
            if (t < 0) return;
            ring_tile_call(*R, t);
        }
    }
};
