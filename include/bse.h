/* bse.h - C ABI of the B200-native screened-exchange hot path of the low-rank BSE method
 * (arxiv 2409.15116, "WEST-BSE").  Citations are PAPER.md line numbers.
 *
 * What the library computes
 *   bse_build_tau : overlap screen of occupied-orbital pairs (eq. 16) and, for every
 *                   surviving pair (v<=v'), the screened Coulomb pair integral
 *                       tau_vv'(r) = int W(r,r') u_v(r') u_v'(r') dr'              (eq. 6)
 *                   with W = v_c + v_c^{1/2} chibar v_c^{1/2} applied through the PDEP low-rank form
 *                       chibar = sum_a |phi_a> lambda_a/(1-lambda_a) <phi_a|       (eq. 9-11)
 *   bse_apply_k1x : out[b,v] = P_c sum_{v'} tau_vv' a[b,v'],  P_c x = x - sum_w u_w <u_w|x>
 *                                                               (eq. 5 and PAPER.md:67; the paper's K^1d)
 *
 * Conventions (normative)
 *   grid n1 x n2 x n3 (this version: n1 = n2 = n3 = n in {12 16 20 24 30 32 36 40 48 60 64 72 80 96 100 108 120 128 144
 *   160}, cubic cell of edge L, else BSE_EUNSUPPORTED),
 *   linear index (i1*n + i2)*n + i3;  r = (L/n) i;  G = (2 pi/L) m;  Hartree atomic units.
 *   sphere S = { m : |m|^2 <= floor(2 ecut (L/2pi)^2 (1+1e-12)) };  R = floor(sqrt(max)) must be < n/2.
 *   half sphere H = { m in S : m3>0 } U { m3=0, m2>0 } U { m3=m2=0, m1>=0 }, sorted by ascending
 *   ((m1 mod n) n + (m2 mod n)) n + (m3 mod n);  Npw_h = |H|.  PW arrays hold c(G) on H, interleaved
 *   (re,im), with f(r) = sum_{G in S} c(G) e^{+iG.r}, c(-G) = conj c(G), c(0) real.
 *   v_c(G) = 4 pi/|G|^2, v_c(0) := 0.  phi_a normalised sum_S |phi_a(G)|^2 = 1, phi_a(0) = 0.
 *   Everything is fp64.
 *
 * Ownership: the caller owns every array it passes.  With device pointers (default) `u` and `phi` are
 *   BORROWED: they must stay alive and unmodified until bse_destroy.  With BSE_PTR_HOST the library copies
 *   them to device memory it owns during bse_create.  `out` must not alias `a`.  The library owns the pair
 *   list, the tau store and all workspaces.
 * Errors: every call returns a status; nothing throws or exits across the ABI.  There is NO CPU fallback:
 *   without a CUDA device every compute entry point returns BSE_ECUDA.
 * Asynchrony: work is enqueued on the cudaStream_t passed at create (NULL = default stream); calls that
 *   return host data synchronise that stream.  bse_build_tau synchronises once (pair count read-back).
 */
#ifndef BSE_H
#define BSE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bse_handle bse_handle;

enum { BSE_OK = 0, BSE_EINVAL = -1, BSE_ENOMEM = -2, BSE_ECUDA = -3, BSE_ESTATE = -4, BSE_EUNSUPPORTED = -5 };

/* flags of bse_create */
#define BSE_TAU_REAL   0x0u   /* tau_vv'(r) stored on the real-space grid, [P][N] doubles (default)          */
#define BSE_TAU_PW     0x1u   /* tau_vv'(G) stored on H, [P][Npw_h] complex; inverse FFT inside the apply     */
#define BSE_TAU_STREAM 0x2u   /* nothing kept between calls: every bse_apply_k1x rebuilds tau(G) in pair batches into
                                 a transient buffer and streams tau(r) from it in row batches                    */
#define BSE_TAU_MASK   0x3u
#define BSE_VEC_REAL   0x0u   /* a/out = [B][Nv][N] real (default)                                            */
#define BSE_VEC_PW     0x4u   /* a/out = [B][Nv][Npw_h] complex on H ("of length N_pw"); a(0) must be
                                 real; out = P_c of (sum_v' tau a) truncated to S.  With BSE_TAU_PW/STREAM the products
                                 are formed on the smallest supported grid n_a >= 3R+1 (alias-free inside S)     */
#define BSE_TAU_F32    0x10u  /* with BSE_TAU_PW / BSE_TAU_STREAM: tau(G) is KEPT as complex64 (each pair integral is computed in fp64 and
                                 rounded once); halves the store and the coefficient sweeps of the apply.  Mixed-precision variant
                                 (PAPER.md:279); results then carry a relative error of about 2^-24 = 6e-8 instead of 1e-15, so the
                                 1e-10 parity bar applies to the default (double) store only.  bse_get_tau returns the unrounded
                                 double values (recomputed) */
#define BSE_PTR_HOST   0x8u   /* u and phi passed to bse_create are HOST pointers (copied to the device)      */

/* Create a problem instance.  Builds the sphere/stick tables, twiddles and v_c^{1/2} on the host and uploads
 * them; launches no heavy work.
 *   grid[3]   n1,n2,n3 (i3 fastest)                cell[9]  row-major lattice vectors (bohr)
 *   ecut      Ha, sphere |G|^2/2 <= ecut           Nv, u    [Nv][N] real, orthonormal: dV sum_r u_v u_w = delta
 *   Npdep,phi [Npdep][Npw_h] complex interleaved on H   lambda [Npdep] HOST pointer, every lambda < 1
 *   eta       overlap threshold of eq. 16: pair kept iff O_vv' >= eta; diagonal always kept
 *   stream    cudaStream_t (as void*) or NULL
 * Errors: BSE_EINVAL (null pointer, non-positive size, lambda >= 1, eta < 0, sphere does not fit: R >= n/2,
 * Npdep > 2(Npw_h-1)), BSE_EUNSUPPORTED (non-cubic cell or grid, odd n, radix other than 2,3,5),
 * BSE_ENOMEM, BSE_ECUDA. */
int bse_create(bse_handle **h, const int grid[3], const double cell[9], double ecut,
               int Nv, const double *u, int Npdep, const double *phi, const double *lambda,
               double eta, unsigned flags, void *stream);

/* Screen (eq. 16) -> pair list; then tau for every listed pair unless BSE_TAU_STREAM.  May be called again
 * (rebuilds).  Errors: BSE_ENOMEM before any work is launched if the tau store does not fit. */
int bse_build_tau(bse_handle *h);

/* out[b,v] = P_c sum_v' tau_vv' a[b,v'] for B trial blocks.  a, out: DEVICE pointers, layout per
 * BSE_VEC_* flag.  BSE_ESTATE if bse_build_tau has not run.  The first call plans its staging buffers from the device
 * memory that is free then (up to 92 % of it: tau(r) row batches, real-space copies of a group of trial blocks) and keeps
 * them; BSE_ENOMEM if one trial block plus one row of pairs does not fit. */
int bse_apply_k1x(bse_handle *h, const double *a, double *out, int B);

/* K1e term of the Liouville operator (eq. 4), same layouts and conventions as bse_apply_k1x:
 *   out[b,v] = 2 P_c [ u_v(r) v_H[b](r) ],  v_H[b](G) = v_c(G) n_b(G) on S (v_c(0) := 0),  n_b(r) = sum_v' u_v'(r) a[b,v'](r).
 * Needs no pair list (may be called before bse_build_tau).  REAL layout: the product u_v v_H is not truncated; PW layout: it
 * is truncated to S before P_c and formed on the apply grid.  K1e - K1x (the caller's sign) is the two-body kernel of eq. 1. */
int bse_apply_k1e(bse_handle *h, const double *a, double *out, int B);

/* Both two-body terms in one call, sharing the transforms of a, the accumulated rows and ONE P_c:
 *   out[b,v] = P_c ( ce * 2 u_v v_H[b]  +  cd * sum_v' tau_vv' a[b,v'] );   eq. 1 uses ce = 1, cd = -1.
 * Equals ce * bse_apply_k1e + cd * bse_apply_k1x (P_c is linear) at about the cost of bse_apply_k1x alone.
 * BSE_ESTATE if bse_build_tau has not run. */
int bse_apply_k1(bse_handle *h, const double *a, double *out, int B, double ce, double cd);

/* Change of representation of trial blocks between the Kohn-Sham and the localised orbitals (eq. 12, PAPER.md:104-106;
 * "a transformation of A_s between the two spaces is necessary"):
 *   transpose == 0: y[b,v,:] = sum_v' U[v][v'] x[b,v',:]      transpose != 0: y[b,v,:] = sum_v' U[v'][v] x[b,v',:]
 * U: DEVICE [Nv][Nv] row-major real orthogonal (Gamma point); x, y: DEVICE, layout per BSE_VEC_* flag; y must not alias x. */
int bse_rotate(bse_handle *h, const double *U, int transpose, const double *x, double *y, int B);

/* JADE localisation of the occupied orbitals (eq. 12-15): the U that bse_rotate applies and
 * that makes the screen of eq. 16 effective.  Needs no handle.
 *   psi     DEVICE [Nv][N] real orthonormal orbitals on the n^3 grid (cubic cell of edge cell[0], even n)
 *   U       DEVICE [Nv][Nv] row-major, written: psi~_v = sum_v' U[v][v'] psi_v' (eq. 12) minimises the spread of eq. 14
 *   psi_loc DEVICE [Nv][N] or NULL: U psi
 *   tol, max_sweeps  sweeps of concurrent Givens rotations (round-robin rounds of disjoint pairs; every angle of a round from
 *           the six matrices A^(n) = <psi|cos,sin(2 pi x/L)|psi> as they stand) until the largest |sin theta| of a sweep < tol
 *   init_eig != 0: start from the eigenvectors of A^(1) sorted by ascending eigenvalue (the paper's choice), else the identity
 *   sweeps  HOST, may be NULL: sweeps done      spread HOST [2], may be NULL: sigma^2 of eq. 14 before and after
 * Work runs on an internal stream ordered after `stream`; `stream` is made to wait for the results; the call synchronises.
 * Readings J1-J4 (angle formula, schedule, stopping, orientation): DESIGN.md section 2. */
int bse_jade(const int grid[3], const double cell[9], int Nv, const double *psi, double *U, double *psi_loc,
             double tol, int max_sweeps, int init_eig, int *sweeps, double *spread, void *stream);

/* Row-sharded operation (PAPER.md:156 and Fig. 2: "we distributed the N_occ orbitals across band groups, using a
 * block distribution scheme"): this handle owns the output rows [v0, v1) of every trial block.  Call before bse_build_tau, which
 * then keeps tau only for the pairs (v, v') that touch an owned row (a pair that straddles two owners is built by both);
 * bse_apply_k1x takes the FULL trial blocks a [B][Nv][Npw_h] (after the all-gather of PAPER.md:156) and writes the owned rows
 * only, out [B][v1 - v0][Npw_h].  u (replicated) and P_c are unchanged.  Needs BSE_VEC_PW with BSE_TAU_PW / BSE_TAU_STREAM
 * (BSE_EUNSUPPORTED otherwise); (0, Nv) restores the unsharded behaviour.  bse_num_pairs / bse_get_pairs still describe the whole
 * list.  paper_2409_15116_b200/sharded.py drives one such handle per rank with torch.distributed. */
int bse_set_rows(bse_handle *h, int v0, int v1);

/* K1e on a row-sharded trial block (eq. 4 sums over all occupied states inside the integral; "communications
 * between band groups are required only when a summation over occupied states is carried out").  PW layout only.
 *   bse_k1e_hartree_partial: vG[b](G) = v_c(G) sum_{v in [v0,v1)} [u_v a_bv](G) on H, from the rows this rank holds
 *       a_rows DEVICE [B][v1-v0][Npw_h] complex;  vG DEVICE [B][Npw_h] complex (written)
 *   the caller sums vG over the ranks (an all-reduce of B * Npw_h coefficients), then
 *   bse_k1e_from_hartree:    out_rows[b, v-v0] = P_c [ 2 u_v v_H[b] ], v_H[b] the potential with coefficients vG[b]
 *       out_rows DEVICE [B][v1-v0][Npw_h] complex (written)
 * With (v0, v1) = (0, Nv) the two calls together are bse_apply_k1e. */
int bse_k1e_hartree_partial(bse_handle *h, const double *a_rows, int v0, int v1, int B, double *vG);
int bse_k1e_from_hartree(bse_handle *h, const double *vG, int v0, int v1, int B, double *out_rows);

/* Same with HOST pointers: copies a to the device, applies, copies out back, synchronises (the end-to-end
 * call bench.py times as `e2e`).  With BSE_TAU_REAL the blocks are pipelined: block b+1 is copied in and block b-1
 * copied out (two copy streams) while block b is applied.  In the other storage modes the copy of a runs on a copy
 * stream while tau is rebuilt (BSE_TAU_STREAM), and every row chunk that P_c has finished is copied out on the second copy
 * stream while the next chunk is projected.  Pinned host memory is needed for the overlap. */
int bse_apply_k1x_host(bse_handle *h, const double *a_host, double *out_host, int B);

/* Replace u and/or phi (either may be NULL) of a handle created with BSE_PTR_HOST by new HOST arrays of the same sizes:
 * host-to-device copy into the buffers the handle owns, nothing reallocated.  The copy is ENQUEUED (a copy stream of the
 * handle, ordered after the work already on its stream) and the call returns: with pinned host memory the arrays must stay
 * unchanged until the next call on this handle that synchronises (bse_build_tau + bse_get_pairs, bse_apply_k1x_host, ...).
 * u goes in column slabs (all orbitals on a range of grid points), and the bse_build_tau that follows screens each slab as
 * it arrives (a1 is a sum over grid points), so the copy hides the screen.  tau is invalidated (call bse_build_tau again).
 * BSE_ESTATE if the handle borrows device arrays. */
int bse_set_inputs_host(bse_handle *h, const double *u_host, const double *phi_host);

int bse_destroy(bse_handle *h);

/* ---- read-only accessors (parity tests, input construction) ---- */
int bse_npw_half(const bse_handle *h, long long *npw_h);
int bse_gvectors(const bse_handle *h, int *mill /* HOST [Npw_h][3] */);
int bse_num_pairs(const bse_handle *h, long long *P);
int bse_get_pairs(const bse_handle *h, int *pairs /* HOST [P][2], lexicographic, v<=v' */);
int bse_get_overlap(const bse_handle *h, double *O /* HOST [Nv][Nv], eq. 16 */);
/* tau of pairs [first, first+count) into a DEVICE buffer; layout BSE_TAU_REAL ([count][N] doubles) or
 * BSE_TAU_PW ([count][Npw_h] complex).  Works in every storage mode (recomputes if needed). */
int bse_get_tau(bse_handle *h, long long first, long long count, double *dst, unsigned layout);

/* ---- allocation-free screen (a1, eq. 16) ----
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it):
 *   M[v][w] = sum_r u_v(r)^2 u_w(r)^2   for v <= w   (the matrix whose normalised form bse_get_overlap returns and
 *   bse_build_tau thresholds against eta), by the same split-K FP64 tensor-core SYRK + reduction as bse_build_tau.
 * It needs no handle and calls no cudaMalloc / cudaFree / allocating library routine: the split-K partial sums go to a
 * fixed array of BSE_SCREEN_STATIC_BYTES (8 MiB) that is part of the library image, so EVERY GPU that loads the library
 * holds those 8 MiB until the process exits, and Nv is limited to BSE_SCREEN_STATIC_MAX_NV = 1024 (8 Nv^2 bytes must fit;
 * the split-K factor is at most floor(8 MiB / (8 Nv^2)), so near the limit the call is correct but slower than the
 * handle's path).  Larger Nv: BSE_EINVAL with a message naming the limit.
 *   u      DEVICE [Nv][N] doubles, 16-byte aligned, N even (BSE_EINVAL otherwise); read only
 *   M      DEVICE [Nv][Nv] doubles, written; entries with v <= w are defined (raw sums, no dV, not normalised), entries
 *          below the diagonal are unspecified (zero, or the symmetric value inside a diagonal 64 x 64 tile)
 *   stream the CUDA stream (cudaStream_t) everything is enqueued on; the call does not synchronise
 * The array is shared by every call of the process on that GPU and keeps the last call's contents: each call clears it first
 * (on `stream`), so calls on the same stream are safe back to back, while calls that overlap on the GPU (different streams,
 * or several host threads) RACE on it: serialise them.  The first call on a device resolves the array's device address
 * (cudaGetSymbolAddress, once per device, with that device current): make that call outside stream capture. */
#define BSE_SCREEN_STATIC_BYTES  (8u << 20)
#define BSE_SCREEN_STATIC_MAX_NV 1024
int bse_screen_overlap_static(const double *u, int Nv, long long N, double *M, void *stream);

/* ---- measurement helpers ---- */
/* Debug / test knobs of one handle (nothing is read from the environment).  They only lower a limit or choose between
 * equivalent kernels, never change a result:  "max_group" caps the number of trial blocks processed together in the PW
 * layout, "max_batch" caps the pairs of one row batch (so that small cases exercise the multi-group / multi-batch paths of
 * the large configurations; 0 = no cap);  "compact_inv" = k forces the compact inverse plane kernel sized for k CTAs per SM
 * (0 = never, -1 = automatic);  "slab_rows" = k caps the rows per chunk of the plane-slab apply (PW layout with tau on H; -1 = never
 * take that path, 0 = no cap), "slab_planes" = k the planes per slab; setting "max_group" or "max_batch" also keeps the apply on the group / row-batch path;
 * "pc_rows" = k caps the rows P_c projects per chunk (0 = no cap); "in_chunks" = k makes bse_set_inputs_host copy u in k
 * column slabs (0 = automatic: 8 from 256 MB on, else 1);  "pipe" picks the plane-pass kernels (1 = the pipelined,
 * bulk-copy staged ones wherever they fit, 0 = the one-plane-per-CTA ones, -1 = automatic: pipelined for the inverse and the
 * single-field forward pass from n = 120 on), "pipe_lc" = k caps the packed lines per slab of the pipelined kernels (0 = no cap).
 * BSE_EINVAL for an unknown key. */
int bse_debug_set(bse_handle *h, const char *key, long long value);
/* Per-stage device time (CUDA events on the library's stream).  enable != 0 switches recording on (adds a
 * host sync per call).  Stage indices: BSE_ST_*; ms and launches are arrays of BSE_ST_COUNT, accumulated since
 * the last bse_profile_reset. */
enum { BSE_ST_SCREEN = 0, BSE_ST_PAIRLIST, BSE_ST_FWD_PLANE, BSE_ST_FWD_STICK, BSE_ST_PROJECT, BSE_ST_BACKPROJECT,
       BSE_ST_INV_STICK, BSE_ST_INV_PLANE, BSE_ST_ACCUM, BSE_ST_PC_OVERLAP, BSE_ST_PC_UPDATE, BSE_ST_K1E_DENSITY,
       BSE_ST_K1E_PRODUCT, BSE_ST_COUNT };
int bse_profile_enable(bse_handle *h, int enable);
int bse_profile_reset(bse_handle *h);
int bse_profile_get(const bse_handle *h, double *ms /* [BSE_ST_COUNT] */, long long *launches /* [BSE_ST_COUNT] */);
/* Algorithmic work of the launches since the last reset (always counted): flops and compulsory HBM bytes per stage,
 * by the per-unit figures of DESIGN.md section 6 times the units each launch processed. */
int bse_profile_model(const bse_handle *h, double *flops /* [BSE_ST_COUNT] */, double *bytes /* [BSE_ST_COUNT] */);
/* Implementation traffic NOT in that model: bytes of the stick-plane intermediate Z handed from one pass of the 3-D transform to
 * the other (it exists only because the transform is two kernels).  bench.py reports fractions with and without it. */
int bse_profile_handoff(const bse_handle *h, double *bytes /* [BSE_ST_COUNT] */);
const char *bse_stage_name(int stage);

/* Device time (ms, CUDA events on the library's stream) of the most recent fill of the tau store - the pair integrals a2..a8
 * (+a9 for BSE_TAU_REAL) of all P pairs, screen and list excluded: inside bse_build_tau for BSE_TAU_REAL / BSE_TAU_PW, inside
 * the apply for BSE_TAU_STREAM (where bse_build_tau only screens).  Synchronises.  BSE_ESTATE if nothing was filled yet. */
int bse_last_tau_fill_ms(bse_handle *h, double *ms);

/* FP64 peak probe: runs a dependent-free DMMA (mma.sync m8n8k4 f64) chain and a DFMA chain on every SM and
 * returns the achieved TFLOP/s of each (the roofline denominators for the dense contractions). */
int bse_probe_fp64_peak(double *dmma_tflops, double *dfma_tflops, void *stream);

const char *bse_last_error(void);
const char *bse_version(void);

#ifdef __cplusplus
}
#endif
#endif /* BSE_H */
