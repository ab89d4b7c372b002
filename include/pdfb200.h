/*
 * pdfb200.h -- C-ABI of libpdfb200: batched parton-distribution and alpha_s interpolation
 * on one NVIDIA B200 (sm_100a), fp64.
 *
 * What the library computes is the hot path of PDFFlow (arXiv:2009.06635; citations are
 * lines of PAPER.md): "a log-bicubic PDF interpolation in terms of x and Q^2" following the
 * LHAPDF6 prescription, on Q^2 sub-grids that are interpolated independently, with one-sided
 * rules "close to quark mass thresholds and grids x edges" (section 2.2), and
 * "a log-cubic interpolation with constant extrapolation from the (alpha_s(Q), Q) nodes",
 * sub-grid aware (section 2.3).  The exact formulas (readings O1-O6) are stated
 * in DESIGN.md; the paper prints none.
 *
 * Conventions
 *   - Every call returns an int: PDFB_OK (0) or a negative PDFB_E* code; pdfb_strerror()
 *     gives text.  No C++ exception crosses this boundary.
 *   - "host" / "device" on a pointer says where the memory lives.  Device pointers must
 *     belong to the device the handle was loaded on.
 *   - Handles own all device memory they allocate until *_free().  *_load() copies its host
 *     arrays; the caller may free them immediately.
 *   - Evaluation calls with device pointers allocate nothing, never synchronise and only
 *     enqueue work on `cuda_stream` (a cudaStream_t passed as void*; NULL = default stream).
 *     They can therefore be captured in a CUDA graph and replayed.
 *   - Evaluation calls on ONE handle may be issued from several host threads and be in flight on
 *     several streams at the same time; *_load() / *_free() / *_host() of a handle must not run
 *     concurrently with other calls on the same handle.  (Batches of at most 65 536 points take one of
 *     64 per-handle slots round robin: keep fewer than 64 of them in flight on one handle.  A call that
 *     is recorded by a stream capture takes its slot from a second ring of 64 that live calls never
 *     use, and keeps it for every replay: a graph may replay next to any live calls, and one handle
 *     serves up to 64 recorded small-batch calls that can run at the same time.)
 *   - A given batch gives bit-identical results run to run.  A query on a knot of the grid returns
 *     the table value bit for bit (readings O3, R-ln), the last knot of either axis included.
 *   - There is no CPU fallback: without a CUDA device *_load() fails with PDFB_ECUDA.
 */
#ifndef PDFB200_H
#define PDFB200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pdfb_grid pdfb_grid;     /* opaque; PDF knot grid on one device   */
typedef struct pdfb_alphas pdfb_alphas; /* opaque; alpha_s node list on one device */

enum {
    PDFB_OK = 0,
    PDFB_EINVAL = -1,   /* null pointer, negative size, bad count                       */
    PDFB_EKNOTS = -2,   /* knots not strictly increasing / non-positive / subgrids do not
                           share their threshold knot / a subgrid has < 2 Q knots        */
    PDFB_EPID = -3,     /* requested PID not in the grid (PID 0 is an alias of 21)       */
    PDFB_ECUDA = -4,    /* CUDA runtime error (no device, out of memory, launch failure) */
    PDFB_EIO = -6,      /* a file could not be opened or read                          */
    PDFB_EFORMAT = -7,  /* a file is not in the expected text layout                   */
    PDFB_EXKNOTS = -8,  /* a well-formed member file / argument list this entry point cannot take:
                           sub-grids with different PID lists; or sub-grids with their own x-knot
                           arrays handed to an entry point that wants one array (use the *_xs one) */
    PDFB_ELIMIT = -5,   /* more than PDFB_MAX_SUBGRIDS subgrids or PDFB_MAX_PIDS PIDs    */
    PDFB_ESTATIC = -9   /* alphas_q2_static: more than PDFB_STATIC_MAX_KNOTS nodes -- the node table
                           would not fit the library's fixed scratch array; use alphas_grid_load */
};
#define PDFB_MAX_SUBGRIDS 16
#define PDFB_MAX_PIDS 32
#define PDFB_MAX_MEMBERS 4096
#define PDFB_LUMI_MAXF 14   /* pdf_lumi_events: at most this many PIDs in the grid */

/*
 * pdf_grid_load -- upload one PDF member's knot grid and run the grid-setup kernel
 * (reading O2: finite-difference derivative rule, one-sided at x edges and at sub-grid
 * edges).
 *
 *   n_sub      number of Q^2 sub-grids, >= 1
 *   nx         number of x knots (shared by all sub-grids), >= 2
 *   x_knots    host [nx], strictly increasing, > 0
 *   q_offsets  host [n_sub+1], q_offsets[0] = 0; sub-grid s owns q_knots[q_offsets[s] ..
 *              q_offsets[s+1]), at least 2 knots each
 *   q_knots    host [q_offsets[n_sub]], Q in GeV (not Q^2), strictly increasing inside a
 *              sub-grid; the last knot of sub-grid s equals the first of s+1 (the threshold)
 *   n_pid,pids host [n_pid], PDG ids of the value columns (e.g. -5..5 and 21)
 *   values     host, xf at the knots, layout [s][ix][iq][ipid] row-major with the sub-grids
 *              concatenated (LHAPDF grid-file order)
 *              (every value must be finite, else PDFB_EINVAL)
 *   device     CUDA device ordinal
 *   out        receives the handle
 */
int pdf_grid_load(int n_sub, int nx, const double *x_knots, const int *q_offsets,
                  const double *q_knots, int n_pid, const int *pids, const double *values,
                  int device, pdfb_grid **out);

/*
 * pdf_grid_load_xs -- a member whose sub-grids carry their OWN x-knot arrays, as the LHAPDF6 grid
 * layout allows (every sub-grid block of a member file has its own x line; the files
 * "are directly loaded", sub-grids are interpolated independently).  The cell, the in-cell
 * coordinate and the x derivatives of a point come from the x knots of the point's own sub-grid;
 * below x_min the value continues from that sub-grid's first two knots.
 *   x_offsets  host [n_sub+1], x_offsets[0] = 0; sub-grid s owns x_knots[x_offsets[s] .. x_offsets[s+1])
 *   x_knots    host, the arrays one after the other, each strictly increasing with >= 2 knots; all
 *              arrays must start at the same x_min and end at the same x_max (else PDFB_EKNOTS)
 *   values     host, [s][ix_s][iq_s][ipid] with the sub-grids concatenated (file order)
 * Other arguments as pdf_grid_load.  If the arrays are in fact identical the handle is an ordinary
 * pdf_grid_load handle; otherwise every call on it is served by the read-only-cache kernel (correct
 * everywhere, about an order of magnitude slower than the shared-memory kernel).
 */
int pdf_grid_load_xs(int n_sub, const int *x_offsets, const double *x_knots, const int *q_offsets,
                     const double *q_knots, int n_pid, const int *pids, const double *values,
                     int device, pdfb_grid **out);

/*
 * pdf_set_load -- a PDF SET: n_members member tables on the same knots (section
 * 4.3 "Multi-PDF members evaluation": all flavours of N_rep members on one batch of points).
 * Arguments as pdf_grid_load, plus
 *   n_members  1 .. PDFB_MAX_MEMBERS
 *   values     host, [member][s][ix][iq][ipid]: each member in LHAPDF grid-file order
 * pdf_grid_load is pdf_set_load with one member; pdf_xfxq2 / pdf_xfxq evaluate member 0.
 */
int pdf_set_load(int n_members, int n_sub, int nx, const double *x_knots, const int *q_offsets,
                 const double *q_knots, int n_pid, const int *pids, const double *values,
                 int device, pdfb_grid **out);

/* Number of members of the handle (0 on NULL). */
int pdf_set_members(const pdfb_grid *g);

/*
 * pdf_xfxq2_members -- members member0 .. member0+n_mem-1 on the SAME n points: every member is
 * the interpolation of pdf_xfxq2 applied to its own table (cell location and weights do not depend
 * on the member).  One launch; allocates nothing, never synchronises.
 *   out    device [n_mem][n_req][n]: out[(m*n_req + r)*n + p] = xf of pids[r], member member0+m, point p
 * PDFB_EINVAL if the member range is not inside the set.  Points with no value are counted once.
 */
int pdf_xfxq2_members(const pdfb_grid *g, int member0, int n_mem, int n_req, const int *pids,
                      long long n, const double *x, const double *q2, double *out, void *cuda_stream);
/* The same with the scale given as Q in GeV (see pdf_xfxq). */
int pdf_xfxq_members(const pdfb_grid *g, int member0, int n_mem, int n_req, const int *pids,
                     long long n, const double *x, const double *q, double *out, void *cuda_stream);

/*
 * pdf_xfxq2 -- xf_pid(x, Q^2) for n points and n_req flavours (section 2.2;
 * readings O3-O5).  Points outside the grid are continued (x < x_min, Q^2 outside
 * [q_min, q_max]); points with no value (x > x_max, x <= 0, Q^2 <= 0, NaN, Inf) give NaN in
 * every flavour and are counted (pdf_grid_status).
 *
 *   pids   host [n_req]; each must be in the grid (else PDFB_EPID, nothing is launched)
 *   x, q2  device [n], fp64, read-only
 *   out    device [n_req][n], flavour-major: out[r*n + p] = xf of pids[r] at point p
 */
int pdf_xfxq2(const pdfb_grid *g, int n_req, const int *pids, long long n, const double *x,
              const double *q2, double *out, void *cuda_stream);

/*
 * pdf_xfxq -- the second interpolating method of the PDF ("interpolating methods
 * (two for the PDF and two for alpha_s)"): the scale is given as Q in GeV.  Defined as
 * pdf_xfxq2(x, Q*Q) with the product rounded once in fp64; Q <= 0 or NaN has no value (NaN,
 * counted).  Same arguments, layout, ownership and errors as pdf_xfxq2.
 *   q      device [n], fp64, Q in GeV
 */
int pdf_xfxq(const pdfb_grid *g, int n_req, const int *pids, long long n, const double *x,
             const double *q, double *out, void *cuda_stream);

/*
 * pdf_xfxq2_host -- the same for HOST buffers (pinned or pageable): chunks are copied to the
 * device, evaluated and copied back on internal streams, overlapping the three stages.
 * Synchronous: returns when `out` is complete.  Staging buffers are owned by the handle.
 */
int pdf_xfxq2_host(pdfb_grid *g, int n_req, const int *pids, long long n, const double *x,
                   const double *q2, double *out);

/* Number of points so far that had no value (synchronises the device; sticky counter). */
int pdf_grid_status(const pdfb_grid *g, long long *n_invalid_points);

/* Device time of the grid-setup kernels of this handle's pdf_grid_load, in ms (-1 on NULL). */
double pdf_grid_setup_ms(const pdfb_grid *g);

/* 1 if pdf_xfxq2 on this handle runs the shared-memory kernel (grid qualifies: nx >= 4, every
 * sub-grid >= 4 Q knots, a 4-column or at least a 2-column slice of the table fits shared memory),
 * 0 if it runs the read-only-cache fallback kernel.  Setting PDFB_FORCE_FALLBACK in the
 * environment before pdf_grid_load forces 0, PDFB_NO_W4 forces the 2-column slices (testing). */
int pdf_grid_uses_smem_path(const pdfb_grid *g);

void pdf_grid_free(pdfb_grid *g);

/*
 * alphas_grid_load -- upload the (Q_k, alpha_s(Q_k)) nodes.
 *   q_knots  host [n_knots], Q in GeV, non-decreasing, > 0; a repeated value marks a flavour
 *            threshold and splits the list into sub-grids (the two copies may carry
 *            different alpha_s); every sub-grid needs >= 2 nodes
 *   alphas   host [n_knots]
 */
int alphas_grid_load(int n_knots, const double *q_knots, const double *alphas, int device,
                     pdfb_alphas **out);

/*
 * alphas_q2 -- alpha_s(Q^2) for n points (reading O6): cubic Hermite in ln Q^2 inside the
 * node range with one-sided derivatives at sub-grid edges, frozen at the first / last node
 * value outside ("constant extrapolation").  Q^2 <= 0 or NaN gives NaN.
 *   q2, out  device [n]
 */
int alphas_q2(const pdfb_alphas *a, long long n, const double *q2, double *out,
              void *cuda_stream);

/* alphas_q -- alpha_s at Q in GeV: alphas_q2(Q*Q), the product rounded once in
 * fp64; Q <= 0 or NaN gives NaN.  q: device [n]; out: device [n]. */
int alphas_q(const pdfb_alphas *a, long long n, const double *q, double *out, void *cuda_stream);

/* alphas_q2 for HOST buffers; synchronous. */
int alphas_q2_host(pdfb_alphas *a, long long n, const double *q2, double *out);

void alphas_grid_free(pdfb_alphas *a);

/*
 * alphas_q2_static -- alphas_q2 for a caller that cannot allocate device memory.
 *
 * Who needs it.  PDFFlow runs inside a TensorFlow process, and a framework of that kind
 * claims almost all of the GPU's memory for its own pool at start-up: a cudaMalloc issued by a side
 * library then fails with "out of memory" however little it asks for.  The same goes for a process on
 * a fixed device-memory quota that is already spent, and for an event loop that cannot take the
 * device-wide synchronisation cudaMalloc / cudaFree bring.  alphas_grid_load allocates (a few KB for
 * the node table it derives); this call does not: no cudaMalloc, no cudaFree, no allocating routine,
 * no handle.  The derived table (ln of the nodes, interval records) goes into ONE fixed array of
 * PDFB_STATIC_SCRATCH_BYTES (22 KB) that is part of the library image.  Every GPU of a process that
 * loads libpdfb200.so holds that array from load to exit, used or not.
 *
 *   n_knots, q_knots, alphas   host arrays, the node list exactly as alphas_grid_load takes it (same
 *                  checks, same codes).  At most PDFB_STATIC_MAX_KNOTS (256) nodes: a longer list is
 *                  refused with PDFB_ESTATIC and nothing is launched -- load it with alphas_grid_load.
 *   n, q2, out     device [n] on the CURRENT device (there is no handle to name one); out[i] is the
 *                  value alphas_q2 gives (reading O6): identical bits when alphas_q2 serves the list by
 *                  its general kernel (more than 192 nodes), within the library's 1e-12 rule when it
 *                  serves it by the table-logarithm kernel.
 *   cuda_stream    the node table is rebuilt on this stream ahead of the evaluation, on every call
 *                  (3 + number of sub-grids small launches); nothing synchronises.
 *
 * Sharing.  All calls on a device use the same array, and it keeps whatever the previous call wrote.
 * A call rewrites every entry it later reads, so nothing needs clearing between calls and a shorter
 * list after a longer one is safe -- but two calls whose work overlaps on the GPU (different streams
 * without an event between them, or two host threads) overwrite each other's table and both results
 * are undefined.  Order them on one stream, or with events.
 *
 * First call.  The first call on a device looks up the array's device address (once per device, with
 * that device current) and the SM count; make that call before starting any stream capture.
 */
#define PDFB_STATIC_MAX_KNOTS 256
#define PDFB_STATIC_SCRATCH_BYTES 22528
int alphas_q2_static(int n_knots, const double *q_knots, const double *alphas, long long n,
                     const double *q2, double *out, void *cuda_stream);

const char *pdfb_strerror(int code);

/*
 * pdf_xfxq2_pm, pdf_xfxq2_f32 -- pdf_xfxq2 with another output layout / precision (
 * the interpolating methods of the PDF object).  Same arguments, same arithmetic (fp64),
 * same error behaviour as pdf_xfxq2; compile-time variants of the same kernels.
 *   pdf_xfxq2_pm   out: device double [n][n_req], point-major: out[p*n_req + r] (all flavours of an
 *                  event next to each other, the layout an event loop reads)
 *   pdf_xfxq2_f32  out: device float [n_req][n], flavour-major: the fp64 result rounded ONCE to fp32 at
 *                  the store (half the output bytes; NaN where no value is defined)
 */
int pdf_xfxq2_pm(const pdfb_grid *g, int n_req, const int *pids, long long n, const double *x,
                 const double *q2, double *out, void *cuda_stream);
int pdf_xfxq2_f32(const pdfb_grid *g, int n_req, const int *pids, long long n, const double *x,
                  const double *q2, float *out, void *cuda_stream);

/*
 * pdf_lumi_events -- the fused call for Monte-Carlo integrands.  An event of a
 * hadron-collider integrand carries the momentum fractions of the two beams and ONE factorisation
 * scale (section 4.1; section 4.2; "events of the order of 10^6
 * at once"); what the integrand needs from the PDF is the parton luminosity
 *
 *   lumi[e] = sum_{t < n_terms} coeff[t] * xf(pid_a[t]; x1[e], q2[e]) * xf(pid_b[t]; x2[e], q2[e])
 *
 * with xf exactly the value pdf_xfxq2 returns (in range and outside the grid alike).  One call
 * replaces pdf_xfxq2(x1), pdf_xfxq2(x2), the caller's contraction and, if `a` is given, alphas_q2 on
 * the same scales: ln Q^2, the Q^2 interval and its weights are taken once per event, and 8 (16)
 * bytes per event are written instead of 176.
 *   a, alphas_out  both NULL, or an alpha_s handle of the same device and a device array [n] that
 *                  receives alpha_s(q2[e])
 *   n_terms, pid_a, pid_b, coeff   host arrays [n_terms]: the flavour-pair table c_ab as a list of
 *                  terms (PID 0 = 21; a pair may appear more than once: coefficients add up); every
 *                  PID must be in the grid (PDFB_EPID), every coefficient finite
 *   x1, x2, q2     device [n]
 *   lumi           device [n]; NaN where either point has no value (x > x_max, x <= 0, Q^2 <= 0, NaN;
 *                  counted by pdf_grid_status, once per event)
 *   flags          bit 0: divide by x1[e] * x2[e] (the luminosity of f = xf / x)
 * Member 0 of a set.  Grids with more than PDFB_LUMI_MAXF PIDs: PDFB_ELIMIT.  Allocates nothing,
 * never synchronises, enqueues two or three kernels on `cuda_stream`.
 */
int pdf_lumi_events(const pdfb_grid *g, const pdfb_alphas *a, int n_terms, const int *pid_a, const int *pid_b,
                    const double *coeff, long long n, const double *x1, const double *x2, const double *q2,
                    double *lumi, double *alphas_out, int flags, void *cuda_stream);

/* Diagnostic: out[i] = the library's coordinate logarithm of in[i] (device pointers, in > 0).
 * Every ln of a knot or of a query coordinate goes through this one function (R-ln). */
int pdfb_debug_ln(const double *in, double *out, long long n, void *cuda_stream);

/* Kernels launched by this library since load (all handles); for bench accounting. */
long long pdfb_launch_count(void);

/*
 * Host-only front-end for grids in the LHAPDF6 text layout that PDFFlow reads (
 * SURVEY.md 8(f).2).  Nothing here touches a device: the arrays go to pdf_grid_load /
 * pdf_set_load / alphas_grid_load.
 *
 * Member file ("lhagrid1"): metadata header, then blocks separated by lines "---"; a block is the
 * x knots (line 1), the Q knots in GeV (line 2), the PIDs (line 3), then nx*nq lines of n_pid
 * values, x index outer, Q index inner -- pdf_grid_load's own order.  All blocks must share one PID
 * list (else PDFB_EXKNOTS, after the file has been read to the end and found well-formed).  Blocks
 * may carry different x-knot arrays: pdfb_lhagrid_dims / _get then return PDFB_EXKNOTS and
 * pdfb_lhagrid_dims_xs / _get_xs (which serve both kinds) give pdf_grid_load_xs's arguments.
 * PDFB_EIO: cannot read; PDFB_EFORMAT: not this layout.  The handle owns host memory until
 * pdfb_lhagrid_free.
 *   pdfb_lhagrid_get fills caller arrays sized from pdfb_lhagrid_dims:
 *   x_knots[nx], q_offsets[n_sub+1], q_knots[nq_tot], pids[n_pid], values[nx*nq_tot*n_pid].
 */
typedef struct pdfb_lhagrid pdfb_lhagrid;
int pdfb_lhagrid_read(const char *path, pdfb_lhagrid **out);
int pdfb_lhagrid_dims(const pdfb_lhagrid *g, int *n_sub, int *nx, int *nq_tot, int *n_pid);
int pdfb_lhagrid_get(const pdfb_lhagrid *g, double *x_knots, int *q_offsets, double *q_knots, int *pids,
                     double *values);
/* x_offsets[n_sub+1], x_knots[nx_total] (the blocks' x arrays one after the other), values[n_values] */
int pdfb_lhagrid_dims_xs(const pdfb_lhagrid *g, int *n_sub, int *nx_total, int *nq_tot, int *n_pid,
                         long long *n_values, int *shared_x);
int pdfb_lhagrid_get_xs(const pdfb_lhagrid *g, int *x_offsets, double *x_knots, int *q_offsets, double *q_knots,
                        int *pids, double *values);
void pdfb_lhagrid_free(pdfb_lhagrid *g);
/* alpha_s nodes of a set's metadata file: the lists AlphaS_Qs (GeV, a repeated Q marks a
 * threshold) and AlphaS_Vals.  *n = node count; the arrays are filled only if cap >= *n. */
int pdfb_lhapdf_info_alphas(const char *info_path, int cap, double *q_knots, double *alphas, int *n);
/* NumMembers of a set's metadata file (1 if the key is absent). */
int pdfb_lhapdf_info_members(const char *info_path, int *n_members);

#ifdef __cplusplus
}
#endif
#endif /* PDFB200_H */
