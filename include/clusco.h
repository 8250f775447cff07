/*
 * clusco.h -- C ABI of the B200-native (sm_100a) cRMSD library.
 *
 * The calls follow the problem statement of the ClusCo paper (arxiv 1302.4000; citations are
 * /root/reference/PAPER.md:<line>): an ensemble of N models of L C-alpha atoms each, equal length
 * and one-to-one atom correspondence (eq. 1 has a single atom index i), is compared
 * all-versus-all -- N(N-1)/2 scores -- or against one reference/native structure
 * (PAPER.md:84, 126-134).  The score is the coordinate RMSD after optimal superposition (eq. 1),
 * obtained WITHOUT a rotation matrix from the 3x3 covariance matrix M of the pair, the eigenvalues of
 * M^T M found as cubic roots, S = sign det M and the two radii of gyration (eq. 2):
 *
 *     cRMSD = sqrt( R_A^2 + R_B^2 - 2 (sqrt(l1) + sqrt(l2) + S sqrt(l3)) ).
 *
 * Conventions for every call
 *   - Pointers are DEVICE pointers unless the name ends in _host.  The caller owns every buffer; the
 *     library keeps no reference after the call is enqueued and frees nothing of the caller's.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Device-pointer
 *     calls are asynchronous on that stream and never synchronise the device.  *_host calls block.
 *   - coords[N][L][3]: float32, row-major, xyz interleaved, Angstrom (any unit; the result is in the
 *     same unit).  Need not be centred.  Base pointers must be 16-byte aligned.
 *   - Return value: clusco_status (0 = OK).  Nothing throws or aborts across the ABI.
 *     N < 0, L < 1, or a NULL pointer with a non-empty extent -> CLUSCO_ERR_INVALID_ARG.
 *     N == 0 (or N < 2 for all-pairs) is valid and writes nothing.
 *   - NaN/Inf coordinates propagate to NaN results for the pairs they touch (no error: the call is
 *     asynchronous).  Results are symmetric by construction; the diagonal is not stored.
 *   - A device that is not compute capability 10.x -> CLUSCO_ERR_UNSUPPORTED_DEVICE.  There is no
 *     CPU fallback.
 *
 * Accuracy of the cRMSD calls, and the domain in which it is claimed (measured against the
 * FP64 oracle by tests/test_gpu_parity.py on every pair of the ensembles named below).  The bar is BASELINE.json's:
 * |c^2 - c^2_exact| <= 2e-3 A^2 for every pair, and |c - c_exact| <= 1e-3 A wherever c_exact >= 0.5 A.
 * c^2 = R_A^2 + R_B^2 - 2E is a difference of numbers of the size of the squared radii of gyration, so the error
 * of every variant is RELATIVE to R_A^2 + R_B^2, not absolute:
 *   - tensor-core engine (CLUSCO_ENGINE_I8TC, the default for L <= 256): coordinates are quantised to 24-bit fixed
 *     point per model (step = 2^-23 x the model's largest centred coordinate, rounded up to a power of two), the
 *     Gram sums of the quantised coordinates are EXACT, the closed form runs in fp32 with a Newton-polished E kept
 *     as an unevaluated pair.  Measured: max |dc^2| = 1.3e-3 A^2 (rms 2.4e-4) over 1.8e7 pairs at R_g^2 = 4289 A^2
 *     (the most extended native of the generator, L = 250), 8.6e-4 at 1693 A^2, 2.5e-4 on C3 (843 A^2); i.e.
 *     max |dc^2| ~ 1.5e-7 (R_A^2 + R_B^2).  The bar is therefore claimed for R_A^2 + R_B^2 <= 9000 A^2 (R_g up to
 *     ~65 A -- more than twice the R_g of any real protein of <= 256 residues); beyond that the error keeps growing
 *     in proportion and the bar is not claimed (use CLUSCO_ENGINE_FFMA through clusco_crmsd_allpairs_ex).
 *   - CUDA-core engine (CLUSCO_ENGINE_FFMA, any L; the default for L > 256): fp32 products in 16-atom blocks, FP64
 *     running totals, FP64 closed form.  Measured max |dc^2| = 6.4e-4 A^2 (rms 1e-4) at R_g^2 = 4289 A^2, i.e.
 *     ~7e-8 (R_A^2 + R_B^2): the bar is claimed for R_A^2 + R_B^2 <= 25 000 A^2.
 *   - one-vs-all: fp32 sums over 8 lanes x L/8 atoms, fp32 closed form; 1.2e-3 A^2 at R_g^2 = 3202 A^2 (L = 150);
 *     same domain as the tensor-core engine.
 * Coordinates in other units scale these figures by the square of the unit.  Per-model scale exponents are clamped
 * to [-30, 30]: a model whose largest centred coordinate is >= 2^30 (or NaN/Inf) yields NaN for its pairs; a model
 * whose largest centred coordinate is below 2^-31 keeps the 2^-53 quantisation step (one bit of its 24 lost per
 * factor of two).  L <= 256 for the
 * tensor-core engine (int32 level sums, A operand resident in tensor memory); N <= 2^24.
 */
#ifndef CLUSCO_H
#define CLUSCO_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    CLUSCO_OK = 0,
    CLUSCO_ERR_INVALID_ARG = 1,
    CLUSCO_ERR_WORKSPACE_TOO_SMALL = 2,
    CLUSCO_ERR_UNSUPPORTED_DEVICE = 3,
    CLUSCO_ERR_CUDA = 4
} clusco_status;

/* Gram-stage engines of the all-pairs kernel.                              */
typedef enum {
    CLUSCO_ENGINE_AUTO = 0,   /* the library's default for this device and shape                      */
    CLUSCO_ENGINE_FFMA = 1,   /* fp32 CUDA-core Gram, 16-atom blocked accumulation                    */
    CLUSCO_ENGINE_I8TC = 2    /* tcgen05 kind::i8 tensor-core Gram on 3x8-bit fixed-point slices,
                                 exact int32 accumulation in TMEM                                     */
} clusco_engine;

/* Static, never freed. */
const char* clusco_status_string(int status);
/* cudaError_t behind the last CLUSCO_ERR_CUDA returned on this host thread (0 if none). */
int clusco_last_cuda_error(void);
/* Library version, "major.minor". */
const char* clusco_version(void);

/* 1 if `engine` can run models of L atoms on the current build, else 0 (host-only query). */
int clusco_engine_supported(int engine, int32_t L);

/*
 * Host-only query: how the tensor-core engine decomposes an (N, L) all-pairs call -- out5 = { tiles of the upper
 * triangle, 32-atom k-steps per tile, MMA columns issued per k-step and tile (all six digit products), row models
 * per tile, column models per tile }.  One tile and k-step costs 128 rows x out5[2] columns x 32 atoms multiply-adds
 * on the tensor pipe; bench.py derives the ISSUED work of its roofline from this (the ALGORITHMIC work is 9 L
 * multiply-adds per pair).  CLUSCO_ERR_INVALID_ARG if the engine does not take L.
 */
int clusco_i8tc_geometry(int64_t N, int32_t L, int64_t* out5);

/*
 * Centring and radius of gyration (implicit in eq. 2: M and R are taken about the centroid,
 * PAPER.md:40-45).   coords[N][L][3] -> centred[N][L][3] = x_i - mean(x)   (same layout; may alias
 * coords; may be NULL), r2[N] = (1/L) sum_i |x_i - mean|^2 = R^2 (may be NULL).
 */
int clusco_center(const float* coords, int64_t N, int32_t L, float* centred, float* r2, void* stream);

/*
 * Workspace for the all-pairs call: bytes of device scratch (operand planes in the Gram stage's
 * layout + per-model scale and sum of squares).  Returns 0 for invalid arguments.
 */
size_t clusco_crmsd_allpairs_workspace(int64_t N, int32_t L);

/*
 * All-versus-all cRMSD (eq. 2 for every pair; N(N-1)/2 values).
 *   out[N(N-1)/2]: row-major packed upper triangle, for i < j
 *       out[ i*(2N-i-1)/2 + (j-i-1) ] = cRMSD(model i, model j).
 *   workspace: >= clusco_crmsd_allpairs_workspace(N, L) bytes, 256-byte aligned, contents undefined
 *       on entry and exit; else CLUSCO_ERR_WORKSPACE_TOO_SMALL.
 */
int clusco_crmsd_allpairs(const float* coords, int64_t N, int32_t L, float* out,
                          void* workspace, size_t workspace_bytes, void* stream);

/*
 * The same with an explicit Gram engine and a row range: computes rows [row_begin, row_end) of the
 * packed triangle -- the contiguous slice
 *       out_rows[ idx(i,j) - idx(row_begin, row_begin+1) ],  row_begin <= i < row_end, j > i
 * -- so that ranks of a multi-GPU job each own one contiguous slice of the matrix and exchange
 * nothing.  row_begin must be a multiple of 128 (or 0) unless row_begin == row_end.
 */
int clusco_crmsd_allpairs_ex(const float* coords, int64_t N, int32_t L,
                             int64_t row_begin, int64_t row_end, float* out_rows,
                             void* workspace, size_t workspace_bytes, int engine, void* stream);

/*
 * The two stages of the all-pairs call, separately (clusco_crmsd_allpairs_ex = prepare + compute on one
 * stream).  prepare: steps a1+a2 -- centroid, power-of-two scale and sum of squares per model, and the
 * operand planes of `engine` -- written into `workspace`.  compute: steps a3-a5 for rows
 * [row_begin,row_end) from a prepared workspace (same N, L, engine; AUTO resolves identically in both).
 * A prepared workspace can serve any number of compute calls (row ranges, repeated timing).
 */
int clusco_allpairs_prepare(const float* coords, int64_t N, int32_t L, void* workspace,
                            size_t workspace_bytes, int engine, void* stream);
int clusco_allpairs_compute(int64_t N, int32_t L, int64_t row_begin, int64_t row_end, float* out_rows,
                            void* workspace, size_t workspace_bytes, int engine, void* stream);

/*
 * Fused consumers of the all-versus-all matrix (the matrix itself is never written to memory).
 *
 * clusco_crmsd_allpairs_below -- the paper's first use case computes all-versus-all cRMSD and keeps the pairs
 * below a cut-off ("awk '{if($3<3.2) ...}'").  Here the filter and the compaction run in the
 * epilogue of the all-pairs kernel:  for every i < j with cRMSD(i,j) < cutoff (compared in fp32 on the value
 * the all-pairs call would store) one triple pair_i[k] = i, pair_j[k] = j, pair_c[k] = cRMSD is written; the
 * order of the triples is unspecified.  *count (device, 8 bytes) receives the number of such pairs; if it
 * exceeds `capacity` the first `capacity` slots are valid and the rest were dropped (call again with more).
 * NaN pairs are never below.  capacity == 0 counts only (the three arrays may then be NULL).
 *
 * clusco_crmsd_rowstats -- the per-model reductions that cluster-representative selection consumes (mean
 * cRMSD of a model to the others, neighbour counts within a cut-off):
 *     rowsum[i] = sum_{j != i} cRMSD(i,j)   (float64; summation order unspecified: atomics),
 *     below[i]  = #{ j != i : cRMSD(i,j) < cutoff }.
 * A NaN/Inf model makes its own rowsum and every other rowsum NaN (it is a term of each).
 *
 * workspace: as clusco_crmsd_allpairs.  Both calls are asynchronous on `stream`.
 */
int clusco_crmsd_allpairs_below(const float* coords, int64_t N, int32_t L, float cutoff, int64_t capacity,
                                int32_t* pair_i, int32_t* pair_j, float* pair_c, unsigned long long* count,
                                void* workspace, size_t workspace_bytes, void* stream);
int clusco_crmsd_rowstats(const float* coords, int64_t N, int32_t L, float cutoff, double* rowsum,
                          int32_t* below, void* workspace, size_t workspace_bytes, void* stream);

/*
 * All-versus-all distance RMSD, the paper's eq. 5:
 *     dRMSD(A,B) = sqrt( 2/(L(L-1)) sum_{i<j} (d_ij^A - d_ij^B)^2 ),  d_ij = |x_i - x_j|
 * (mirror images score 0: "loses chirality").  out[N(N-1)/2]: the same packed row-major upper
 * triangle as clusco_crmsd_allpairs.  Computed as one tensor-core Gram contraction over the K = L(L-1)/2
 * distances per model, in exact 3 x 8-bit fixed point; needs 2 <= L <= 296 (int32 accumulators), L = 1 gives
 * all zeros, L > 296 -> CLUSCO_ERR_INVALID_ARG.  workspace: >= clusco_drmsd_allpairs_workspace(N, L) bytes
 * (about 3 N K bytes: the int8 distance planes), 256-byte aligned.  NaN/Inf coordinates propagate to NaN
 * for the pairs of that model.  Asynchronous on `stream`.
 */
size_t clusco_drmsd_allpairs_workspace(int64_t N, int32_t L);
int clusco_drmsd_allpairs(const float* coords, int64_t N, int32_t L, float* out,
                          void* workspace, size_t workspace_bytes, void* stream);

/*
 * All-versus-all contact map overlap, the paper's eq. 6-7: with the binary contact map
 *     C_ij = 1 if |x_i - x_j| < cutoff else 0      (i < j: contacts are pairs of distinct atoms; the paper gives
 *                                                   no cut-off value, so it is an argument),
 * the Sorensen similarity index  S = 100 * 2 n(A and B) / (n(A) + n(B)),  n(.) = number of contacts.
 * out[N(N-1)/2]: packed row-major upper triangle, S in [0, 100].  Two maps with no contact at all are identical
 * maps: S = 100 (0/0 is read that way; also every pair when L = 1).  The contact decision is taken in FP64 on the
 * fp32 coordinates (sqrt(dx^2 + dy^2 + dz^2) < (double)cutoff, IEEE operations), the counts are exact integers
 * (0/1 int8 operands, int32 tensor-core accumulation), S = (float)(200.0 * n_AB / (n_A + n_B)).
 * Needs L <= 296 (shared-memory staging of a model), cutoff >= 0.  workspace: >= clusco_cmo_allpairs_workspace(N, L)
 * bytes (about N L(L-1)/2 bytes), 256-byte aligned.  NaN/Inf coordinates -> NaN for that model's pairs.
 */
size_t clusco_cmo_allpairs_workspace(int64_t N, int32_t L);
int clusco_cmo_allpairs(const float* coords, int64_t N, int32_t L, float cutoff, float* out,
                        void* workspace, size_t workspace_bytes, void* stream);

/*
 * One reference structure against N models: native[L][3], coords[N][L][3]
 * (neither pre-centred) -> out[N], out[k] = cRMSD(native, model k).
 */
int clusco_crmsd_one_vs_all(const float* native, const float* coords, int64_t N, int32_t L,
                            float* out, void* stream);

/*
 * dRMSD (eq. 5) and contact map overlap (eq. 6-7) of N models against ONE reference structure ("... or with respect to
 * the reference model"): out[n] = the measure of (native, model n), defined as in the
 * all-versus-all calls above (same readings, same contact decision; CMO is bit-exact).  Single pass, FP64, one warp
 * per model; 1 <= L <= 1024 (L = 1: dRMSD 0, CMO 100); cutoff >= 0.  NaN/Inf coordinates -> NaN for that model.
 */
int clusco_drmsd_one_vs_all(const float* native, const float* coords, int64_t N, int32_t L, float* out, void* stream);
int clusco_cmo_one_vs_all(const float* native, const float* coords, int64_t N, int32_t L, float cutoff, float* out,
                          void* stream);

/*
 * GDT_TS, TM-score and MaxSub of N models against one reference structure (eq. 3-4), by the paper's
 * search: every continuous fragment of length 4, L/4, L/2 and L seeds a superposition of the whole model (optimal
 * rigid fit of the fragment); the atoms closer than 3.5 A are superposed again "until the number of selected atoms
 * does not change in four iterations"; after every superposition
 *     C_x = number of atom pairs below x = 1, 2, 4, 8 A,   TM = (1/L) sum_i 1 / (1 + (d_i/d0)^2),
 *     d0 = 1.24 cbrt(L - 15) - 1.8 (clamped at 0.5 A);  MaxSub: the same with d0 = 3.5 A
 * are evaluated and the maxima kept.  out[N][3] (float32): out[3n] = GDT_TS = 100 * (max C_1 + max C_2 + max C_4 +
 * max C_8) / (4 L) in percent, out[3n+1] = TM-score, out[3n+2] = MaxSub.  native[L][3], coords[N][L][3], neither
 * pre-superposed.  Readings of the points the paper leaves open (duplicate fragment lengths, iteration cap of 20,
 * at least 3 selected atoms, strict inequalities): DESIGN.md section 14.  The search is data dependent, so the
 * kernel works in FP64 throughout.  3 <= L <= 1024.  NaN/Inf coordinates give NaN for that model.
 */
int clusco_gdt_one_vs_all(const float* native, const float* coords, int64_t N, int32_t L, float* out, void* stream);
/*
 * The same three scores all-versus-all: out[N(N-1)/2][3], packed row-major upper triangle as in
 * clusco_crmsd_allpairs; for the pair i < j model i plays the reference (the search is symmetric in the two
 * structures -- selections depend on distances only -- so the scores are those of (j, i) too).  One warp per pair;
 * the cost is ~5 us of FP64 work per pair at L = 150, so this is meant for thousands of models, not millions.
 */
int clusco_gdt_allpairs(const float* coords, int64_t N, int32_t L, float* out, void* stream);

/*
 * Host-buffer calls (blocking; the end-to-end path): coords_host / native_host / out_host are ordinary host
 * pointers -- pinned (page-locked) memory lets the transfers overlap the kernels, pageable memory works
 * but serialises.  Device scratch (inputs, result, workspace) is taken from a library-owned
 * stream-ordered memory pool that is KEPT between calls, so a repeated call pays no allocation;
 * transfers run on the library's own copy stream:
 *   all-pairs:   H2D coords -> prepare -> for each of 8 row chunks of equal pair count
 *                (clusco_partition_rows): compute chunk k | D2H chunk k-1;
 *   one-vs-all:  the models go up in ~64 MB chunks, each scored as soon as it has landed.
 * One host call runs at a time per process (internal lock).  Errors: as the device calls, plus
 * CLUSCO_ERR_CUDA for allocation / copy failures (nothing is leaked; the streams are drained first).
 */
int clusco_crmsd_allpairs_host(const float* coords_host, int64_t N, int32_t L, float* out_host);
int clusco_crmsd_one_vs_all_host(const float* native_host, const float* coords_host, int64_t N,
                                 int32_t L, float* out_host);
/*
 * Host-buffer forms of the two fused consumers (the paper's first use case end to end, and the
 * per-model reductions of PAPER.md:116): coordinates go up, only the triples / the per-model statistics come down --
 * at C3 (10 000 x 250) 30 MB up and 18 MB down instead of the 200 MB matrix.  Semantics as
 * clusco_crmsd_allpairs_below / clusco_crmsd_rowstats; every pointer is a HOST pointer (count_host too); blocking;
 * same pool, lock and error behaviour as the calls above.  `capacity` may be a generous bound (up to N(N-1)/2): the
 * device staging starts at 4 Mi triples and the compute stage is run a second time, with room for all, only when
 * more pairs than that were found and the caller has room for them.  *count_host = number of pairs found (may exceed
 * capacity: the first `capacity` triples are valid).
 */
int clusco_crmsd_allpairs_below_host(const float* coords_host, int64_t N, int32_t L, float cutoff, int64_t capacity,
                                     int32_t* pair_i_host, int32_t* pair_j_host, float* pair_c_host,
                                     unsigned long long* count_host);
int clusco_crmsd_rowstats_host(const float* coords_host, int64_t N, int32_t L, float cutoff, double* rowsum_host,
                               int32_t* below_host);
/* Returns the pool kept by the *_host calls to the driver and destroys their streams (all devices). */
int clusco_host_release(void);

/*
 * Balanced row partition for `parts` ranks: writes parts+1 boundaries (multiples of 128, first 0,
 * last N) such that each [b[r], b[r+1]) owns about the same number of pairs.  Host-only arithmetic.
 */
int clusco_partition_rows(int64_t N, int32_t parts, int64_t* boundaries_host);

#ifdef __cplusplus
}
#endif
#endif /* CLUSCO_H */
