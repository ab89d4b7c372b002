// xfxq2_smem.cu -- K2/K3, the shared-memory path of pdf_xfxq2 (readings O3-O5).
//
// Why it looks the way it does ("Kernel design"): per point and flavour the method
// gathers a 4x4 value stencil -- 1408 B of table per point at 11 flavours against 104 B of HBM
// traffic -- and the points of a warp almost never share a cell.  The gather is what bounds the
// kernel, so it is fed from shared memory at full crossbar width, with no bank conflict:
//   * the value table is split into FLAVOUR GROUPS of 4 columns; one group's slice
//     [iq][ix4][4] (32 B per knot, iq over the concatenated Q^2 knots) fits shared memory and is
//     staged once per CTA by TMA bulk copies.  Each persistent CTA serves one group for all
//     points of its tiles, so it writes whole flavour rows with coalesced stores and no point
//     ever has to be re-ordered;
//   * the 4x4 stencil is always read as 4 consecutive rows x 4 consecutive knots, rows i-1..i+2 of
//     the concatenated table.  In an edge interval the stencil reaches one row / one knot outside
//     the knot array or the sub-grid; that knot carries weight exactly 0 (one-sided derivative
//     rule, reading O2), so whatever finite number sits there contributes nothing: a neighbouring
//     sub-grid's row, the next row's first knot, or the interval records that bracket the slice in
//     shared memory.  Rows are a uniform stride apart, so the 32 loads of a point use 8 per-lane
//     addresses + 3 uniform offsets (LDS [R+UR]) and no address arithmetic;
//   * one window row (4 knots x 4 flavours) is 128 contiguous bytes = 8 chunks of 16 B that
//     cover all 8 bank groups.  Lane l reads them in the rotated order c = (s + l - 2*node0) & 7,
//     so at every step the 8 lanes of a quarter-warp hit 8 distinct bank groups whatever cells
//     their points fell in: 32 conflict-free LDS.128 per point and group, 4 wavefronts each;
//   * the x weights are rotated the same way (selects on the ALU pipe), so no data is moved back.
// Knot location uses a uniform-in-log lookup table corrected by comparisons on the raw knots
// (the result is defined by the comparisons, reading Q5).
#include <atomic>
#include <cstdlib>

#include "xfxq2_slow.cuh"

#define PDFB_RR_CACHE_MAX 8192  // SETS: batches up to this size keep their points' (cell, t, tau) in shared memory (24 B each)

template <int MODE, int W>  // compile-time (xfxq2_smem.cuh): a run-time flag costs 11 % (register pressure at the 128 cap)
__global__ void __launch_bounds__(NT_SMEM, 1)
k_xfxq2_smem(const __grid_constant__ GridDev g, const __grid_constant__ PassList pl, long long n,
             const double *__restrict__ x, const double *__restrict__ q2, double *__restrict__ out,
             long long out_stride, int member0, int n_req, int n_jobs, const int *__restrict__ row_range)
{
    constexpr bool Q_IS_Q = MODE & 1;
    constexpr int OUT = (MODE >> 1) & 3;
    constexpr bool SETS = (MODE >> 3) & 1;  // persistent over jobs: more (member, pass) jobs than SMs
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) unsigned long long mbar[2];  // the rows of buffer 0 / 1 have landed
    __shared__ unsigned char wcnt[NT_SMEM / 32][8];  // entries in each warp's class lists
    __shared__ __align__(16) unsigned char s_req[NT_SMEM / 32];  // "evaluate your full batches now", one flag per warp
    const int tid = threadIdx.x, lane = tid & 31;
    // job = (member of the set, pass).  Few jobs: blockIdx.x = seq * n_jobs + job, a job's CTAs share its
    // tiles.  SETS: CTA b takes jobs b, b + gridDim.x, ... over all tiles, the next job's rows in flight.
    int job = SETS ? blockIdx.x : blockIdx.x % n_jobs;
    const int seq = SETS ? 0 : blockIdx.x / n_jobs, nseq = SETS ? 1 : gridDim.x / n_jobs;
    double *const out_base = out;
    const uint32_t tab0 = (uint32_t)__cvta_generic_to_shared(smem) + (uint32_t)g.pre_bytes;
    const uint32_t mb = (uint32_t)__cvta_generic_to_shared(&mbar[0]);
    const int slice_bytes = (W == 4) ? g.slice_bytes : g.slice2_bytes;
    // small batches stage only the table rows their Q^2 values can touch (k_row_range below), at the
    // rows' own places in the slice: nothing else of this kernel changes.  SETS: if twice that many rows
    // fit, the odd jobs of a CTA use a second copy `shift` bytes further up (no point is outside the
    // grid then, k_row_range: the out-of-grid classes, which locate the table themselves, never run).
    const int RBs = (W == 4) ? g.nx4 * 32 : g.nx2 * 16;
    const int r0 = row_range ? row_range[0] : 0, r1 = row_range ? row_range[1] : g.nq_tot;
    const int lo = r0 * RBs, stage = (r1 - r0) * RBs;
    int shift = 0;
    if (SETS && row_range) {
        // even: the copy keeps the bank alignment of 2-column rows.  With r0 == 0 the stencils of Q^2
        // intervals 0 and 1 reach below row 0 with weight exactly 0: row -1, and (x interval 0 of Q^2
        // interval 0: knot -1 of row -1) the tail of row -2.  For buffer 0 that is the tail of `pre`;
        // for buffer 1 it is what lies below its row 0 -- so two rows are left free between the two
        // buffers there and zero-filled below (no bulk copy ever writes them).
        const int rows = (r1 - r0 + (r0 == 0 ? 3 : 1)) & ~1;
        if ((rows + r1) * RBs <= slice_bytes) shift = rows * RBs;
    }
    auto stage_job = [&](int j, int buf) {  // one thread: the rows of job j into buffer buf
        const int ps = j % pl.n, mm = j / pl.n;
        const uint32_t bar = mb + 8u * buf;
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(stage) : "memory");
        const unsigned char *src = reinterpret_cast<const unsigned char *>(W == 4 ? g.valg : g.valg2) +
                                   ((size_t)(member0 + mm) * (W == 4 ? g.n_groups : g.n_groups2) + pl.group[ps]) * slice_bytes + lo;
        for (int o = 0; o < stage; o += 32768) {
            int bytes = min(32768, stage - o);
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"(tab0 + buf * shift + lo + o), "l"(src + o), "r"(bytes), "r"(bar) : "memory");
        }
    };

    // ---- stage this CTA's flavour-group slice with TMA bulk copies; small tables by plain loads
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mb));
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mb + 8u));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (tid < NT_SMEM / 32 * 8) (&wcnt[0][0])[tid] = 0;
    if (tid < NT_SMEM / 32) s_req[tid] = 0;
#ifdef PDFB_CHECKED
    {   // poison the whole window: whatever is read later must have been staged
        uint32_t size;
        asm("mov.u32 %0, %%dynamic_smem_size;" : "=r"(size));
        for (uint32_t e = tid; e < size / 8; e += NT_SMEM) reinterpret_cast<unsigned long long *>(smem)[e] = 0x7ff8dead00000000ULL;
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
#endif
    __syncthreads();
    if (tid == 0) stage_job(job, 0);
    if (SETS && shift && r0 == 0) {  // the two free rows below buffer 1 (see `rows` above): finite data for zero-weight reads
        for (int e = tid; e < 2 * RBs / 16; e += NT_SMEM)
            asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(tab0 + (uint32_t)(shift - 2 * RBs + e * 16)), "r"(0) : "memory");
    }
    {   // pre and post blocks around the slice (both multiples of 128 bytes)
        const int4 *src = reinterpret_cast<const int4 *>(g.aux);
        int4 *pre = reinterpret_cast<int4 *>(smem), *post = reinterpret_cast<int4 *>(smem + g.pre_bytes + slice_bytes);
        const int npre = g.pre_bytes / 16, npost = g.post_bytes / 16;
        for (int e = tid; e < npre; e += NT_SMEM) pre[e] = __ldg(src + e);
        for (int e = tid; e < npost; e += NT_SMEM) post[e] = __ldg(src + npre + e);
    }
    __syncthreads();
    // SETS on a small batch (row range known, no point outside the grid): every job of this CTA sees the
    // SAME points, so the part of a point's evaluation that does not depend on the member table -- both
    // logarithms, both searches, t and tau -- is done once per CTA and kept in the part of the slice area
    // that the staged rows leave free: {t, tau} (16 B) and {x interval, Q^2 row} (8 B) per point.  A job
    // then fetches the two interval records, forms the weights and gathers; results are bit-identical to
    // the loop below (same lane, same arithmetic).
    uint32_t cache = 0, cache_i = 0;  // shared addresses of the two arrays; 0 = no cache
    if constexpr (SETS) {
        if (row_range && r1 - r0 < g.nq_tot && n <= PDFB_RR_CACHE_MAX) {
            const int cbytes = (((int)n * 24) + 127) & ~127;
            const int top = ((shift ? shift + r1 * RBs : lo + stage) + 127) & ~127;
            int cbase = -1;
            if (top + cbytes <= slice_bytes) cbase = top;          // above the rows of both buffers
            else if (cbytes <= lo) cbase = 0;                        // below them
            if (cbase >= 0) {
                cache = tab0 + (uint32_t)cbase;
                cache_i = cache + (uint32_t)(((int)n * 16 + 15) & ~15);
                const SmemViews sv = make_views<W>(g, smem);
                const int lane8 = tid & 7;
                for (int p = tid; p < (int)n; p += NT_SMEM) {
                    const double xs = __ldg(x + p), qs = load_scale<Q_IS_Q>(q2 + p);
                    double tx = 0.0, tq = 0.0;
                    int i = -1, gi = 0;  // i < 0: the point has no value (k_row_range: none is outside the grid)
                    if (xs >= g.x_min && xs <= g.x_max && qs >= g.q2_min && qs <= g.q2_max) {
                        const double u = ln_pos(xs), v = ln_pos(qs);
                        i = locate_x(g, sv, xs, u);
                        gi = locate_q(g, sv, qs, v);
                        const IntervalRec32 rx = load_rec4(sv.xrec + (uint32_t)i * 128u, lane8);
                        const IntervalRec32 rq = load_rec4(sv.qrec + (uint32_t)gi * 128u, lane8);
                        tx = (u - rx.z0) * rx.inv_dz; tq = (v - rq.z0) * rq.inv_dz;
                    }
                    PDFB_ASSERT(cache_i + (uint32_t)p * 8u + 8u <= tab0 + (uint32_t)slice_bytes);
                    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(cache + (uint32_t)p * 16u), "d"(tx), "d"(tq) : "memory");
                    asm volatile("st.shared.v2.s32 [%0], {%1, %2};" ::"r"(cache_i + (uint32_t)p * 8u), "r"(i), "r"(gi) : "memory");
                }
                __syncthreads();
            }
        }
    }
    int jj = 0;
    do {  // jobs of this CTA (one, unless SETS)
    const int buf = shift ? (jj & 1) : 0;
    // (the buffer of job jj - 1 is free: every warp passed the barrier at the end of that job)
    if (SETS && shift && tid == 0 && job + (int)gridDim.x < n_jobs) stage_job(job + gridDim.x, buf ^ 1);
    {
        uint32_t done = 0;
        const uint32_t parity = shift ? ((jj >> 1) & 1) : (jj & 1);
        while (!done)
            asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                         : "=r"(done) : "r"(mb + 8u * buf), "r"(parity) : "memory");
    }
    const int pass = job % pl.n, mem = job / pl.n;
    // (the members of a set follow each other in `out`; fp32 output counts in floats)
    out = (OUT == PDFB_OUT_FM32) ? reinterpret_cast<double *>(reinterpret_cast<float *>(out_base) + (long long)mem * n_req * out_stride)
                                 : out_base + (long long)mem * n_req * out_stride;
    const uint32_t tab = tab0 + (uint32_t)(buf * shift);
    const SmemViews sv = make_views<W>(g, smem);
    const int lane8 = tid & 7;
    const uint32_t RB = sv.row_bytes, rb2 = 2u * RB, rb3 = 3u * RB;
    const bool odd = lane8 & 1;
    const int row[4] = {pl.row[pass][0], pl.row[pass][1], pl.row[pass][2], pl.row[pass][3]};
    const double qnan = __longlong_as_double(0x7ff8000000000000LL);
    // Out-of-grid points are not evaluated where they occur.  Each warp appends their indices to one
    // list per continuation class (xfxq2_slow.cuh) and evaluates them in whole batches of 32, so that
    // every call is class-uniform on full lanes; a remainder stays at the front of its list, so batch
    // k of a class is always the warp's entries 32k .. 32k+31 of that class, whenever it is evaluated
    // (results do not depend on timing).  WHEN: a warp whose list reaches PDFB_SLOW_TRIGGER entries
    // raises a request flag for every warp of the CTA; a warp that holds entries looks at its flag once
    // per tile and then evaluates its full batches -- all warps run the out-of-grid code at about the
    // same time, without a barrier (a barrier every few tiles costs the in-range loop 7-25 %, measured).
    // The lists live in a global scratch slot owned by this SM: at most one CTA of this kernel is
    // resident per SM, on any stream, because the launcher requests more than half of the SM's shared
    // memory (checked at load: occupancy == 1).
    auto wlist = [&]() -> uint32_t * {  // recomputed where needed: nothing of this lives in a register across the hot loop
        uint32_t smid;
        asm("mov.u32 %0, %%smid;" : "=r"(smid));
        return g.slow_ws + ((size_t)(smid % PDFB_WS_SLOTS) * (NT_SMEM / 32) + (threadIdx.x >> 5)) * (PDFB_SLOW_CLASSES * PDFB_SLOW_LCAP);
    };
    constexpr int TILE = NT_SMEM * PPT_SMEM;
    auto flush_lists = [&](bool final) {  // warp-uniform
        flush_warp_lists<MODE, W>(final, wlist(), &wcnt[threadIdx.x >> 5][0], &s_req[threadIdx.x >> 5], &g, smem, x, q2, out, out_stride, n_req, pl.row[pass]);
    };

    if (SETS && cache) {  // the points' table-independent part comes from the cache (above)
        for (int p = tid; p < (int)n; p += NT_SMEM) {
            const double2 tt = lds128(cache + (uint32_t)p * 16u);
            const int2 cell = lds64i(cache_i + (uint32_t)p * 8u);
            const int i = cell.x, gi = cell.y;
            double y[W];
            if (i >= 0) {
                const IntervalRec32 rx = load_rec4(sv.xrec + (uint32_t)i * 128u, lane8);
                const IntervalRec32 rq = load_rec4(sv.qrec + (uint32_t)gi * 128u, lane8);
                double wu[4], vw[4];
                weights_rec32(rx, tt.x, wu);
                weights_rec32(rq, tt.y, vw);
                eval_stencil<W>(tab, RB, rb2, rb3, gi - 1, i - 1, wu, vw, lane8, y);
            } else {
#pragma unroll
                for (int c = 0; c < W; c++) y[c] = qnan;
                if (job == 0) atomicAdd(g.n_invalid, 1ULL);
            }
            store_cols<W, OUT>(out, out_stride, n_req, p, row, y);
        }
    } else {
    bool pending = false;  // this warp has list entries (the flush request is only looked at then)
    // software pipeline: the next tile's coordinates are in flight while this tile is evaluated
    long long tile = seq;
    double xv[PPT_SMEM], qv[PPT_SMEM];
#pragma unroll
    for (int k = 0; k < PPT_SMEM; k++) {
        const long long p = tile * TILE + k * NT_SMEM + tid;
        xv[k] = (p < n) ? __ldg(x + p) : 1.0; qv[k] = (p < n) ? load_scale<Q_IS_Q>(q2 + p) : 1.0;
    }
    while (tile * TILE < n) {
    // the hot loop is left to evaluate class lists (no call inside it: its registers are at the cap)
    for (; tile * TILE < n; tile += nseq) {
        const long long p0 = tile * TILE + tid;
        double xn[PPT_SMEM], qn[PPT_SMEM];
        bool in_range[PPT_SMEM];
        bool any_in = false;
#pragma unroll
        for (int k = 0; k < PPT_SMEM; k++) {
            const long long pn = p0 + k * NT_SMEM + (long long)nseq * TILE;
            xn[k] = (pn < n) ? __ldg(x + pn) : 1.0; qn[k] = (pn < n) ? load_scale<Q_IS_Q>(q2 + pn) : 1.0;
            in_range[k] = (p0 + k * NT_SMEM < n) && xv[k] >= g.x_min && xv[k] <= g.x_max && qv[k] >= g.q2_min && qv[k] <= g.q2_max;
            any_in |= in_range[k];
        }
        if (any_in) {
            // ---- locate (LUT guess + exact comparisons where needed), weights, one gather per point.
#pragma unroll
            for (int k = 0; k < PPT_SMEM; k++) {
                const double xs = in_range[k] ? xv[k] : g.x_min, qs = in_range[k] ? qv[k] : g.q2_min;
                const double u = ln_pos(xs), v = ln_pos(qs);
                const int i = locate_x(g, sv, xs, u);
                const int gi = locate_q(g, sv, qs, v);
                const IntervalRec32 rx = load_rec4(sv.xrec + (uint32_t)i * 128u, lane8);
                const IntervalRec32 rq = load_rec4(sv.qrec + (uint32_t)gi * 128u, lane8);
                double wu[4], vw[4], y[W];
                weights_rec32(rx, (u - rx.z0) * rx.inv_dz, wu);
                weights_rec32(rq, (v - rq.z0) * rq.inv_dz, vw);
                if (W == 4) {  // written out: the register allocation of this path is at the 128 cap
                    Win w;
                    make_win(w, tab + (uint32_t)((gi - 1) * (int)RB), i - 1, wu, lane8);
                    double2 E, O;
                    gather4(w, vw, RB, rb2, rb3, E, O);
                    y[0] = odd ? O.x : E.x; y[1] = odd ? O.y : E.y; y[W - 2] = odd ? E.x : O.x; y[W - 1] = odd ? E.y : O.y;
                } else {
                    eval_stencil<W>(tab, RB, rb2, rb3, gi - 1, i - 1, wu, vw, lane8, y);
                }
                if (in_range[k]) store_cols<W, OUT>(out, out_stride, n_req, p0 + k * NT_SMEM, row, y);
            }
        }
#pragma unroll
        for (int k = 0; k < PPT_SMEM; k++) {
            const long long p = p0 + k * NT_SMEM;
            const bool live = p < n;
            const bool invalid = live && !in_range[k] && (!(xv[k] > 0.0) || !(qv[k] > 0.0) || !(xv[k] <= g.x_max) || isinf(qv[k]));
            const bool slow = live && !in_range[k] && !invalid;
            if (invalid) {
                double nanv[W];
#pragma unroll
                for (int c = 0; c < W; c++) nanv[c] = qnan;
                store_cols<W, OUT>(out, out_stride, n_req, p, row, nanv);
                if (job == 0) atomicAdd(g.n_invalid, 1ULL);
            }
            const unsigned slow_mask = __ballot_sync(0xffffffffu, slow);
            if (slow_mask) {  // warp-uniform: append the out-of-grid points to the warp's class lists
                if (slow) {
                    const bool low_x = xv[k] < g.x_min, high_q = qv[k] > g.q2_max, low_q = qv[k] < g.q2_min;
                    const int cls = low_x ? (high_q ? 3 : (low_q ? 4 : 0)) : (high_q ? 1 : 2);
                    const unsigned peers = __match_any_sync(slow_mask, cls);  // the lanes of this class
                    unsigned char *cnt = &wcnt[threadIdx.x >> 5][cls];
                    const int cur = *cnt, kc = __popc(peers);
                    // (cur + kc <= TRIGGER - 1 + 32 + 31 < LCAP: the trigger below empties the list at the end of its tile)
                    PDFB_ASSERT(cur + kc <= PDFB_SLOW_LCAP && p < n);
                    __stcg(wlist() + cls * PDFB_SLOW_LCAP + cur + __popc(peers & ((1u << lane) - 1u)), (uint32_t)p);
                    __syncwarp(slow_mask);
                    if ((peers & ((1u << lane) - 1u)) == 0) {  // the first lane of the class
                        *cnt = (unsigned char)(cur + kc);
                        // a list reaching the trigger length asks every warp of the CTA to evaluate its batches
                        if (cur < PDFB_SLOW_TRIGGER && cur + kc >= PDFB_SLOW_TRIGGER)
                            *reinterpret_cast<uint4 *>(s_req) = make_uint4(0x01010101u, 0x01010101u, 0x01010101u, 0x01010101u);
                    }
                }
                pending = true;  // (looked at together with the request flag; cleared by the flush)
            }
            xv[k] = xn[k]; qv[k] = qn[k];
        }
        if (pending && *reinterpret_cast<volatile unsigned char *>(&s_req[threadIdx.x >> 5])) { tile += nseq; break; }
    }
    if (pending) { flush_lists(false); pending = false; }
    }
    flush_lists(true);
    }
    if (SETS) {
        __syncthreads();  // every warp is done with this job's rows (measured: mbarrier hand-over between the warps
                          // instead of this barrier changes nothing -- a job is bound by its five tile iterations)
        if (!shift && tid == 0 && job + (int)gridDim.x < n_jobs) stage_job(job + gridDim.x, 0);  // one buffer: stage now
    }
    ++jj;
    } while (SETS && (job += gridDim.x) < n_jobs);
}

// Rows of the concatenated Q^2 knot list that a batch can touch: the intervals of its smallest and
// largest in-range Q^2, two rows below and three above (the 4-row stencils and their zero-weight
// overreach); the whole table as soon as one point lies outside the grid (the out-of-grid classes read
// fixed rows at either end and locate the table themselves).  One CTA; for batches small enough that
// staging the whole 200 KB slice per CTA costs as much as evaluating them (PDF sets on an x-grid at
// one scale: 2415 points, 6 rows of 64).
template <bool Q_IS_Q>
__global__ void __launch_bounds__(1024) k_row_range(const GridDev g, long long n, const double *__restrict__ x,
                                                    const double *__restrict__ q2, int *__restrict__ rr)
{
    __shared__ double smin[32], smax[32];
    __shared__ int sout[32];
    double lo = g.q2_max, hi = g.q2_min;
    int outside = 0;
    for (long long p = threadIdx.x; p < n; p += 1024) {
        const double q = load_scale<Q_IS_Q>(q2 + p), xv = x[p];
        if (!(xv > 0.0) || !(xv <= g.x_max) || !(q > 0.0) || isinf(q)) continue;  // no value: touches no row
        if (q >= g.q2_min && q <= g.q2_max) { lo = fmin(lo, q); hi = fmax(hi, q); }
        if (q < g.q2_min || q > g.q2_max || xv < g.x_min) outside = 1;
    }
    for (int o = 16; o; o >>= 1) {
        lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o)); hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
        outside |= __shfl_xor_sync(0xffffffffu, outside, o);
    }
    if ((threadIdx.x & 31) == 0) { smin[threadIdx.x >> 5] = lo; smax[threadIdx.x >> 5] = hi; sout[threadIdx.x >> 5] = outside; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 32; w++) { lo = fmin(lo, smin[w]); hi = fmax(hi, smax[w]); outside |= sout[w]; }
        int r0 = 0, r1 = g.nq_tot;
        if (!outside && lo <= hi) {
            int a = 0, b = 0;  // intervals of lo and hi: the last knot <= the value (a threshold: its upper copy)
            for (int m = 1; m < g.nq_tot; m++) { if (g.q2k[m] <= lo) a = m; if (g.q2k[m] <= hi) b = m; }
            b = min(b, g.nq_tot - 2);
            // rows a-1 .. b+2 hold the stencils; knot -1 of a row is the tail of the row below and knot nx of a
            // row the head of the row above (weight exactly 0, but they must be staged, finite data): one more each
            r0 = max(a - 2, 0); r1 = min(b + 4, g.nq_tot);
        } else if (!outside) { r1 = 1; }  // no point with a value: nothing to stage but a row of finite data
        rr[0] = r0; rr[1] = r1;
    }
}

// Dynamic shared memory of a launch.  Never less than PDFB_SMEM_FLOOR (more than half of the SM's
// 228 KB): two CTAs of this kernel can then not be resident on one SM, whatever the grid size, the
// register count or the stream -- the invariant the per-SM scratch slot of the class lists rests on.
static const int PDFB_SMEM_FLOOR = 116 * 1024;
static const long long PDFB_RR_MAX_POINTS = 65536;  // batches up to this size look for their row range first ...
static const int PDFB_RR_MIN_SLICE = 64 * 1024;      // ... if a slice is at least this big
static int smem_image(const GridDev &d, int W) { return d.pre_bytes + (W == 4 ? d.slice_bytes : d.slice2_bytes) + d.post_bytes; }
static int smem_needed(const GridDev &d, int W) { const int b = smem_image(d, W); return b > PDFB_SMEM_FLOOR ? b : PDFB_SMEM_FLOOR; }
static const int STATIC_SMEM = 256;  // >= the kernel's static shared memory (mbarrier, list counters)
static_assert(NT_SMEM == 512, "PDFB_WS_BYTES and the request flags assume 16 warps per CTA");
static_assert(PDFB_SLOW_TRIGGER - 1 + 32 + 31 <= 255 && PDFB_SLOW_TRIGGER + 62 <= PDFB_SLOW_LCAP, "8-bit list counters");

// %nsmid as the device itself reports it: the class-list scratch is indexed by %smid, and PTX promises
// %smid < %nsmid, not %smid < the SM count of the runtime's device properties.
static __device__ unsigned g_nsmid;
__global__ void k_read_nsmid()
{
    unsigned v;
    asm("mov.u32 %0, %%nsmid;" : "=r"(v));
    g_nsmid = v;
}
static int device_nsmid(int device)  // the caller has made `device` current (pdf_set_load); -1 on error
{
    static std::atomic<int> cached[64];
    if (device < 0 || device >= 64) return -1;
    int v = cached[device].load(std::memory_order_acquire);
    if (v > 0) return v;
    unsigned h = 0;
    k_read_nsmid<<<1, 1>>>();
    pdfb_count_launch(1);
    if (cudaMemcpyFromSymbol(&h, g_nsmid, sizeof(h)) != cudaSuccess || h == 0) { cudaGetLastError(); return -1; }
    cached[device].store((int)h, std::memory_order_release);
    return (int)h;
}

// bit 0: the 4-column slices fit the device's shared memory, bit 1: the 2-column slices do
int pdfb_smem_eligible(const pdfb_grid *g)
{
    if (getenv("PDFB_FORCE_FALLBACK")) return 0;  // testing: force the read-only-cache path
    if (g->sms > PDFB_WS_SLOTS) return 0;         // one scratch slot per SM ...
    const int nsmid = device_nsmid(g->device);    // ... indexed by %smid < %nsmid (read from the device, not assumed = the SM count)
    if (nsmid < 1 || nsmid > PDFB_WS_SLOTS) return 0;
    int dev_max = 0;
    if (cudaDeviceGetAttribute(&dev_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, g->device) != cudaSuccess) return 0;
    int ok = 0;
    if (smem_needed(g->d, 4) + STATIC_SMEM <= dev_max && !getenv("PDFB_NO_W4")) ok |= 1;  // (testing: 2-column path only)
    if (smem_needed(g->d, 2) + STATIC_SMEM <= dev_max) ok |= 2;
    if (!ok) return 0;
    // the attribute is per function, not per handle: raise it once to the device maximum
    static std::atomic<unsigned long long> attr_done{0};  // one bit per device; setting twice is harmless
    const unsigned long long bit = 1ULL << (g->device & 63);
    if (!(attr_done.load(std::memory_order_acquire) & bit)) {
        const int lim = dev_max - STATIC_SMEM;
        cudaError_t e = cudaSuccess;
#define PDFB_ATTR(M, WW) if (e == cudaSuccess) e = cudaFuncSetAttribute(k_xfxq2_smem<M, WW>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim)
        PDFB_ATTR(0, 4); PDFB_ATTR(1, 4); PDFB_ATTR(2, 4); PDFB_ATTR(4, 4);
        PDFB_ATTR(0, 2); PDFB_ATTR(1, 2); PDFB_ATTR(2, 2); PDFB_ATTR(4, 2);
        PDFB_ATTR(8, 4); PDFB_ATTR(9, 4); PDFB_ATTR(8, 2); PDFB_ATTR(9, 2);
#undef PDFB_ATTR
        if (e != cudaSuccess) {
            cudaGetLastError();
            return 0;
        }
        attr_done.fetch_or(bit, std::memory_order_release);
    }
    // the scratch-slot invariant, checked rather than assumed: one resident CTA per SM
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_xfxq2_smem<0, 4>, NT_SMEM, PDFB_SMEM_FLOOR) != cudaSuccess || occ != 1) {
        cudaGetLastError();
        return 0;
    }
    return ok;
}

// passes of a request on W-column groups: one per (group, distinct use of its columns); a PID asked
// for twice gets an extra pass
static int build_passes(int W, int n_groups, int n_req, const int *cols, PassList &pl)
{
    pl.n = 0;
    bool used[PDFB_MAX_PIDS] = {false};
    for (int left = n_req; left > 0;) {
        for (int grp = 0; grp < n_groups && left > 0; grp++) {
            int row[4] = {-1, -1, -1, -1}, hit = 0;
            for (int r = 0; r < n_req; r++)
                if (!used[r] && cols[r] / W == grp && row[cols[r] % W] < 0) { row[cols[r] % W] = r; used[r] = true; hit++; }
            if (!hit) continue;
            if (pl.n >= PDFB_MAX_PIDS) return PDFB_ELIMIT;
            pl.group[pl.n] = grp;
            for (int k = 0; k < 4; k++) pl.row[pl.n][k] = row[k];
            pl.n++;
            left -= hit;
        }
    }
    return PDFB_OK;
}

int pdfb_launch_xfxq2_smem(const pdfb_grid *g, int n_req, const int *cols, long long n, const double *x,
                           const double *q2, double *out, long long out_stride, cudaStream_t st, int mode,
                           int member0, int n_mem)
{
    // Width: a 4-column pass costs ~5.6 shared-memory wavefronts per point (4 gather + 1.6 setup and
    // I/O), a 2-column pass ~3.6; take the cheaper plan among the widths that fit shared memory.
    PassList pl4, pl2;
    pl4.n = pl2.n = 0;
    const int ok = g->d.smem_ok;
    int rc = PDFB_OK;
    if (ok & 1) rc = build_passes(4, g->d.n_groups, n_req, cols, pl4);
    if (!rc && (ok & 2)) rc = build_passes(2, g->d.n_groups2, n_req, cols, pl2);
    if (rc) return rc;
    const bool use2 = !(ok & 1) || ((ok & 2) && 3.6 * pl2.n < 5.6 * pl4.n);
    const PassList &pl = use2 ? pl2 : pl4;
    const int W = use2 ? 2 : 4;
    const int sms = g->sms;
    // jobs = (member, pass).  Few jobs: the SMs are split between them and each CTA is persistent
    // over its share of the tiles.  More jobs than SMs: one CTA per job over all tiles, scheduled
    // by the hardware as SMs free up (one CTA per SM at a time: the slice fills shared memory).
    const long long n_jobs = (long long)pl.n * n_mem;
    if (n_jobs > 0x3fffffff) return PDFB_ELIMIT;
    const int smem = smem_needed(g->d, W);
    // small batch on a big slice: find the rows it needs first (one more launch of a single CTA)
    const int *rr = nullptr;
    if (n <= PDFB_RR_MAX_POINTS && (W == 4 ? g->d.slice_bytes : g->d.slice2_bytes) >= PDFB_RR_MIN_SLICE) {
        // A call recorded by a stream capture keeps the slot chosen here for every replay of its graph: it
        // takes one from a ring of its own, which live calls never use (a replay running next to any
        // number of live calls cannot meet one of them in a slot).
        cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(st, &cap) != cudaSuccess) { cudaGetLastError(); cap = cudaStreamCaptureStatusNone; }  // (legacy stream next to a capture)
        pdfb_grid *gm = const_cast<pdfb_grid *>(g);
        const unsigned idx = (cap == cudaStreamCaptureStatusActive)
                                 ? PDFB_RR_SLOTS + gm->rr_cap_next.fetch_add(1, std::memory_order_relaxed) % PDFB_RR_CAP_SLOTS
                                 : gm->rr_next.fetch_add(1, std::memory_order_relaxed) % PDFB_RR_SLOTS;
        int *slot = g->d.row_range + 2 * idx;
        if (mode & 1) k_row_range<true><<<1, 1024, 0, st>>>(g->d, n, x, q2, slot);
        else k_row_range<false><<<1, 1024, 0, st>>>(g->d, n, x, q2, slot);
        pdfb_count_launch(1);
        rr = slot;
    }
    // the class lists hold point indices as 32-bit offsets: batches beyond 2^31 points go out in slices
    const long long SLICE = 1LL << 31;
    for (long long off = 0; off < n; off += SLICE) {
        const long long m = (n - off < SLICE) ? (n - off) : SLICE;
        int per_job = (int)(sms / n_jobs);
        if (per_job < 1) per_job = 1;
        const long long tiles = (m + NT_SMEM * PPT_SMEM - 1) / (NT_SMEM * PPT_SMEM);
        if (per_job > tiles) per_job = (int)tiles;
        // more jobs than SMs (PDF sets): one persistent CTA per SM walks the jobs, the next job's rows in flight
        const bool sets = n_jobs > sms && mode <= 1;
        const unsigned grid = sets ? (unsigned)sms : (unsigned)(per_job * n_jobs);
#define PDFB_LAUNCH(M, WW) k_xfxq2_smem<M, WW><<<grid, NT_SMEM, smem, st>>>(g->d, pl, m, x + off, q2 + off, out_off, out_stride, member0, n_req, (int)n_jobs, rr)
        // element offset of this slice in `out` (doubles, or floats for the fp32 variant)
        const long long eo = (mode >> 1) == PDFB_OUT_PM64 ? off * n_req : off;
        double *out_off = (mode >> 1) == PDFB_OUT_FM32 ? reinterpret_cast<double *>(reinterpret_cast<float *>(out) + eo) : out + eo;
        if (sets) {
            if (W == 4) { if (mode == 0) PDFB_LAUNCH(8, 4); else PDFB_LAUNCH(9, 4); }
            else        { if (mode == 0) PDFB_LAUNCH(8, 2); else PDFB_LAUNCH(9, 2); }
        } else if (W == 4) { if (mode == 0) PDFB_LAUNCH(0, 4); else if (mode == 1) PDFB_LAUNCH(1, 4); else if (mode == 2) PDFB_LAUNCH(2, 4); else PDFB_LAUNCH(4, 4); }
        else        { if (mode == 0) PDFB_LAUNCH(0, 2); else if (mode == 1) PDFB_LAUNCH(1, 2); else if (mode == 2) PDFB_LAUNCH(2, 2); else PDFB_LAUNCH(4, 2); }
#undef PDFB_LAUNCH
        pdfb_count_launch(1);
    }
    PDFB_CUDA(cudaGetLastError());
    return PDFB_OK;
}
