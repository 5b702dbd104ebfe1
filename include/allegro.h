/* allegro.h — C-ABI boundary of the B200-native Allegro energy+force hot path.
 *
 * What the calls compute is defined by PAPER.md:93 (Allegro hyper-parameters: tensor features, l,
 * full O(3), two-body / latent / edge-energy MLPs, radial cutoff), Table 1,
 * PAPER.md:29 (the architecture of the paper's ref. 22), PAPER.md:9 (strictly local, E(3)-equivariant)
 * and PAPER.md:89/:116 (explicit reversible integrator, 0.48-0.5 fs steps), with every convention the
 * paper leaves open fixed by the readings A1-A24 of SURVEY.md section 8c (listed in DESIGN.md).
 *
 * Conventions
 *  - Every function returns an int status: ALLEGRO_OK (0) or a negative ALLEGRO_ERR_* code.  No C++
 *    exception crosses the boundary.  allegro_last_error(h) returns a NUL-terminated message owned by
 *    the handle (valid until the next call on that handle); with h == NULL it returns the message of
 *    the last failed allegro_create on this thread.
 *  - Pointers marked DEVICE are CUDA device pointers, pointers marked HOST are host pointers.  The
 *    caller owns every array it passes; the library never frees nor retains a caller pointer past the
 *    call.  The handle owns all internal device buffers (neighbour list, workspaces, MD state).
 *  - `stream` is a cudaStream_t passed as void* (NULL = default stream).  Work is enqueued on that
 *    stream; allegro_build_neighbors, allegro_energy_forces, allegro_md_step and the get_* calls
 *    synchronise the stream once before returning so that the status reflects device-side error flags.
 *    There is no host synchronisation inside the step loop of allegro_md_step except the one-word
 *    read-back that sizes a rebuilt neighbour list.
 *  - Units: Angstrom, fs, amu, eV.  Positions / velocities / masses / cell are fp64; the network runs
 *    in fp32.  A cell is a HOST fp64 [3,3] matrix whose ROWS are the lattice vectors a_1, a_2, a_3 (right-handed, det > 0;
 *    else ALLEGRO_ERR_INVALID): orthorhombic (diagonal) or general / triclinic (reading A27 of DESIGN.md).  A
 *    periodic image is x + s_1 a_1 + s_2 a_2 + s_3 a_3; cutoff + skin must not exceed the smallest perpendicular width of the
 *    cell (the box lengths of an orthorhombic cell; ALLEGRO_ERR_CUTOFF).  Only the spatial decomposition (allegro_decomp_select)
 *    still needs an orthorhombic cell.
 *  - There is no CPU fallback: without a CUDA device every compute call returns ALLEGRO_ERR_CUDA.
 */
#ifndef ALLEGRO_B200_H
#define ALLEGRO_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
  ALLEGRO_OK = 0,
  ALLEGRO_ERR_INVALID = -1,      /* bad argument / hyper-parameters / weight count                   */
  ALLEGRO_ERR_UNSUPPORTED = -2,  /* lmax > 3, a row longer than the kernel cap, decomposition of a triclinic cell */
  ALLEGRO_ERR_CUDA = -3,         /* CUDA runtime error (message has the cudaGetErrorString text)       */
  ALLEGRO_ERR_STALE_LIST = -4,   /* some atom moved more than skin/2 since allegro_build_neighbors     */
  ALLEGRO_ERR_NONFINITE = -5,    /* NaN/Inf detected in E or F                                         */
  ALLEGRO_ERR_CUTOFF = -6,       /* r_cut + skin exceeds the smallest box length (reading A17)         */
  ALLEGRO_ERR_SPECIES = -7,      /* a species index outside [0, n_species)                             */
  ALLEGRO_ERR_NO_LIST = -8,      /* energy_forces / get_neighbors before build_neighbors               */
  ALLEGRO_ERR_ALLOC = -9         /* device allocation failed                                           */
};

/* kinds of tensors in the weight blob, as reported by allegro_weight_layout */
enum { ALLEGRO_WK_MATRIX = 0, ALLEGRO_WK_RESIDUAL = 1, ALLEGRO_WK_SIGMA = 2, ALLEGRO_WK_MU = 3 };

/* Hyper-parameters (Table 1).  *_dims lists the output width of each linear layer of the
 * MLP ("dimensions [a,b,c]" = in->a->b->c with SiLU between, none after the last, no biases: A5); the
 * last two_body and latent widths must both equal the latent width D (A10).  edge_dims are the hidden
 * widths of the edge-energy MLP (no non-linearity, final ->1 implicit).  full_o3 = 1 is the paper's
 * "full O(3) symmetry"; 0 keeps only paths with l1+l2+lo even. */
typedef struct {
  int32_t n_species, n_bessel, poly_p, lmax, n_layers, n_channels, full_o3;
  int32_t two_body_nl, two_body_dims[8];
  int32_t latent_nl, latent_dims[8];
  int32_t edge_nl, edge_dims[8];
  double r_cut, avg_num_neighbors;
} allegro_hparams;

/* Layout of the flat fp32 weight blob for `hp` (SURVEY.md 8b "Weight blob order"): tensor t has
 * kind[t] (ALLEGRO_WK_*), rows[t] x cols[t] values, row-major [out,in], tensors concatenated in order.
 * Returns the number of tensors (>= 0) or a negative error; writes at most `max_tensors` entries
 * (arrays may be NULL to query the count only).  HOST pointers.  Pure host logic, no CUDA needed. */
int allegro_weight_layout(const allegro_hparams* hp, int32_t* kind, int64_t* rows, int64_t* cols, int max_tensors);

/* Build a model: validates hp, derives the irreps/path plan and the real coupling tables, copies the
 * weights (HOST pointer, n_weights floats in blob order) to the device.  *handle_out receives the handle. */
int allegro_create(const float* weights_host, size_t n_weights, const allegro_hparams* hp, void** handle_out);
int allegro_destroy(void* h);

/* Row a-1: device cell-list neighbour builder.  pos DEVICE fp64 [N,3] (unwrapped), species DEVICE int32
 * [N], cell HOST fp64 [3,3].  Builds the sorted CSR list of all ordered (i, j, s) with
 * |r_j + s.cell - r_i|^2 < (cutoff+skin)^2 evaluated in fp64 as dx = (x_j-x_i) + ((s_1*a_1x + s_2*a_2x) + s_3*a_3x)
 * (= (x_j-x_i)+s_x*L_x bit for bit when the cell is diagonal), d2=dx*dx+dy*dy+dz*dz (A16, A27), (i,j,s) != (i,i,0), each row
 * sorted by (j, s_1, s_2, s_3).  cutoff must equal hp.r_cut. */
int allegro_build_neighbors(void* h, const double* pos, const int32_t* species, int64_t N,
                            const double* cell, double cutoff, double skin, void* stream);

/* Rows a-2..a-5: energy and forces with the list of the last allegro_build_neighbors.
 * E_out DEVICE fp64 [1]; F_out DEVICE fp64 [N,3]; E_atom_out DEVICE fp32 [N] or NULL.
 * Returns ALLEGRO_ERR_STALE_LIST (outputs undefined) if an atom moved more than skin/2 since the build
 * (with skin = 0 any displacement is stale); it never rebuilds silently. */
int allegro_energy_forces(void* h, const double* pos, const int32_t* species, int64_t N, const double* cell,
                          double* E_out, double* F_out, float* E_atom_out, void* stream);

/* Row a-6: velocity-Verlet NVE (kick-drift-kick, A20), state kept inside the handle.
 * md_init copies pos/vel/mass/species (DEVICE), builds the list and evaluates the initial forces.
 * md_step advances n_steps; after each drift it rebuilds the list when max_i |r_i - r_i^build| > skin/2
 * (skin = 0: every step, A22). */
int allegro_md_init(void* h, const double* pos, const double* vel, const double* mass, const int32_t* species,
                    int64_t N, const double* cell, double cutoff, double skin, void* stream);
int allegro_md_step(void* h, double dt_fs, int64_t n_steps, void* stream);

/* the protocols the paper runs (NVT at 300 K: PAPER.md:49, :116; heating 300 -> 1200 K: :75; tensile strain
 * at fixed rates: :69).  PAPER.md names no thermostat and no deformation scheme; readings A25 / A26:
 *  - allegro_md_step_nvt: velocity-Verlet as allegro_md_step plus Berendsen weak coupling after the second half-kick of step
 *    k = 1..n_steps of this call: T_inst = 2 E_kin / ((3N-3) kB), T_target = T0 + (T1-T0) min(1, k/n_ramp) (n_ramp = 0: T1 at
 *    once), v <- v sqrt(1 + (dt/tau)(T_target/T_inst - 1)).  tau_fs >= dt_fs.  Deterministic; no host sync in the loop.
 *  - allegro_md_deform: affine remap of the unwrapped positions to cell_new (HOST fp64 [3,3]), x' = x L'/L (x' = x H^-1 H' when
 *    either cell is triclinic: the fractional coordinates are kept), full
 *    list rebuild and force evaluation.  A strain rate is a sequence of such increments between allegro_md_step calls.
 *  - allegro_set_state: checkpoint / resume — new pos, vel (DEVICE fp64 [N,3]) for the masses, species and cell given to
 *    allegro_md_init; rebuilds the list and the forces (NVE is deterministic given this state).
 *  - allegro_virial: W[a][b] = -sum_e (rvec_e)_a (dE/d rvec_e)_b [eV] (DEVICE fp64 [9], row-major) from the per-edge gradients
 *    of the LAST force evaluation, with pos (DEVICE) the positions of that evaluation or NULL for the MD state.  The potential
 *    part of the stress is -W / V.  Fixed-order fp64 reduction (deterministic). */
int allegro_md_step_nvt(void* h, double dt_fs, int64_t n_steps, double T0, double T1, int64_t n_ramp, double tau_fs, void* stream);
int allegro_md_deform(void* h, const double* cell_new, void* stream);
int allegro_set_state(void* h, const double* pos, const double* vel, void* stream);
int allegro_virial(void* h, const double* pos, double* W_out, void* stream);

/* Test hook: on = 0 makes the many-channel networks (n = 64) run the forward tensor product and the channel mixing as separate
 * kernels with the per-path products T in HBM (k_tpo_fwd + one GEMM per output irrep) instead of the fused kernel of tp_mix.cu
 * (default, on = 1).  Same arithmetic, other summation order: tests compare the two. */
int allegro_debug_set_fusion(void* h, int on);

/* allegro_virial for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): same arguments, same quantity (the summation order of the fp64 reduction differs, so the last bits may), but
 *  - the call contains no cudaMalloc / cudaFree / allocating library routine and no stream synchronisation: two kernel launches
 *    on `stream`, asynchronous; W_out is valid once the stream has reached that point, and an execution error surfaces at the
 *    caller's next synchronisation;
 *  - the block partials live in a fixed 288 KB file-scope __device__ array (held by every GPU that loads the library until the
 *    process exits), which bounds the size: N > ALLEGRO_VIRIAL_NOALLOC_MAX_ATOMS returns ALLEGRO_ERR_UNSUPPORTED with a message
 *    naming the limit (use allegro_virial then);
 *  - every call on a device shares that array: calls that OVERLAP on the GPU (different streams or handles) race; calls on one
 *    stream are safe.  The array keeps the last call's contents; every entry a call reads it has written first.
 * The handle's device must be the current device on the first call per device (allegro_create does that call's set-up). */
#define ALLEGRO_VIRIAL_NOALLOC_MAX_ATOMS 1048576
int allegro_virial_noalloc(void* h, const double* pos, double* W_out, void* stream);

/* spatial decomposition of the strictly local model (the property behind the paper's 0.964
 * parallel efficiency on Aurora).  One process per GPU; coordinates are replicated on every rank, so the only collective of a
 * step is one all-reduce of the force array and the 8-byte energy (paper_2502_06073_b200/distributed.py).
 *  - allegro_energy_forces_owned: as allegro_energy_forces, but only atoms [0, n_owned) are centre atoms; atoms [n_owned, N) are
 *    ghosts (neighbours only).  E = sum of E_i over the owned atoms, F_out [N,3] = -dE/dr of that partial sum for EVERY atom
 *    (ghost rows hold the reaction forces that the owner rank adds up).
 *  - allegro_decomp_select: local atom set of the brick `coord` of the rank grid `grid` (HOST int32 [3] each): owned atoms first
 *    (wrapped position inside the brick in every decomposed dimension, ascending atom index), then every periodic image within
 *    r_halo of the brick.  Writes local_pos DEVICE fp64 [cap,3] (coordinates inside the local box), local_species DEVICE int32
 *    [cap] (may be NULL), local_src DEVICE int64 [cap] (global atom index), counts HOST int64 [2] = {n_owned, n_local},
 *    local_cell HOST fp64 [3,3] (periodic as the global cell in undecomposed dimensions, padded and pair-free across its wrap in
 *    decomposed ones).  Needs brick + 2 r_halo <= L in decomposed dimensions (an atom appears at most once per rank).
 *  - allegro_decomp_scatter: F_global [N,3] = 0, then F_global[local_src[k]] = F_local[k] (conflict-free, deterministic).
 *  - allegro_kick_drift: v += dt/2 a; if (drift) r += dt v on caller arrays (DEVICE fp64), a = 9.648533212e-3 F / m (A20). */
int allegro_energy_forces_owned(void* h, const double* pos, const int32_t* species, int64_t N, const double* cell, int64_t n_owned,
                                double* E_out, double* F_out, float* E_atom_out, void* stream);
int allegro_decomp_select(void* h, const double* pos, const int32_t* species, int64_t N, const double* cell, const int32_t* grid,
                          const int32_t* coord, double r_halo, int64_t cap, double* local_pos, int32_t* local_species, int64_t* local_src,
                          int64_t* counts, double* local_cell, void* stream);
int allegro_decomp_scatter(const double* F_local, const int64_t* local_src, int64_t n_local, double* F_global, int64_t N, void* stream);
int allegro_kick_drift(double* pos, double* vel, const double* F, const double* mass, int64_t N, double dt_fs, int drift, void* stream);

/* Copies the MD state out.  pos/vel/F DEVICE fp64 [N,3]; E_pot/E_kin DEVICE fp64 [1]; n_rebuilds HOST
 * int64 [1].  Any pointer may be NULL. */
int allegro_get_state(void* h, double* pos, double* vel, double* F, double* E_pot, double* E_kin,
                      int64_t* n_rebuilds, void* stream);

/* Copies the current list out.  E_list HOST int64 [1] is always written (call with the arrays NULL to
 * size them); rowptr DEVICE int64 [N+1], col DEVICE int32 [E_list], shift DEVICE int8 [E_list,3]. */
int allegro_get_neighbors(void* h, int64_t* rowptr, int32_t* col, int8_t* shift, int64_t* E_list);

/* Counters of the last energy_forces / md_step call (HOST int64 [8]): [0] active edges (r < r_cut) of
 * the last force evaluation, [1] list edges, [2] kernel launches of the call, [3] rebuilds of the call,
 * [4] force evaluations of the call, [5] atom chunks per force evaluation (the activation workspace is sized from the
 * free device memory; chunks are exact because the model is strictly local), [6] capacity recoveries of the last md_step (a
 * device-side rebuild outgrew the list: the integrator halts, the host regrows the list and finishes the call — same
 * trajectory), [7] reserved. */
int allegro_get_stats(void* h, int64_t* stats);

/* Per-kernel-class timing for bench.py's roofline line.  allegro_profile(h, 1) resets the counters and makes
 * every launch of the following calls bracketed by CUDA events on the launching stream; allegro_profile(h, 0)
 * stops it.  allegro_get_profile synchronises and returns, per class k (0 gemm, 1 tp_fwd, 2 tp_bwd, 3 gamma,
 * 4 gammabar, 5 active_edges, 6 edge_misc, 7 neighbor, 8 md, 9 force_gather, 10 gemm_f16s, 11 tp_mix, 12 tp_mix16; class 0 = the
 * 3xTF32 kernels of gemm_tc.cu, class 10 = the split-fp16 kernel of gemm_f16s.cu, classes 11 and 12 carry only work: the
 * channel-mixing flop that tensor-product kernels timed in classes 1-2 run on tensor cores themselves (11: mma.sync 3xTF32 in the
 * few-channel kernels, 12: tcgen05 split-fp16 in tp_mix.cu)): ms[k] total device time, launches[k], work[k] =
 * algorithmic flop per active edge summed over the class's launches (classes 0-2, 10-12, else 0).
 * HOST arrays of max_classes entries; returns the number of classes.  Never enabled inside a timed throughput run. */
int allegro_profile(void* h, int enable);
int allegro_get_profile(void* h, double* ms, int64_t* launches, double* work, int max_classes);

/* Debug taps for the CPU-only tests (pure host logic, no CUDA): the library's own real coupling tensor
 * C^(l1 l2 l3) (reading A9), dense row-major [2l1+1][2l2+1][2l3+1] into out (HOST, fp64); and the number of
 * tensor-product paths of layer L (1-based) of the plan derived from hp.  Negative return = error. */
int allegro_debug_coupling(int l1, int l2, int l3, double* out);
int allegro_debug_num_paths(const allegro_hparams* hp, int layer);

/* Test hooks for the split-fp16 tcgen05 GEMM of the wide linears (csrc/gemm_f16s.cu; PAPER.md:93 / Table 1 MLPs).
 * allegro_debug_set_precision: 3 (default) = the full split a_hi b_hi + a_hi b_lo + a_lo b_b (3 x TF32 hi*hi + hi*lo + lo*hi in the
 * chained kernels), 2 = activations split only, 1 = one plain pass — the 1/2-pass kinds exist only for the committed precision
 * study (R4, profiles/r2_precision.md).
 * allegro_debug_gemm runs one launch of that kernel on caller data:  C[M,N] = epi( pro([A0 | A1]) B ),  B(k,n) = wtrans ?
 * W[k*ldw+n] : W[n*ldw+k];  pro / epi are the PRO_* / EPI_* codes of csrc/gemm.cuh (0/1/2 and 0..6).  All pointers DEVICE fp32;
 * A0 / A1 hold rows_cap >= M rows; geo is the [M][8] edge record (u at [4]) or NULL.  Synchronises the stream.
 * Returns ALLEGRO_ERR_UNSUPPORTED when the shape or alignment is outside what the kernel takes.
 * The kernel's packed copy of W is cached by (address, shape): right for the product, whose weights never move or change; a
 * caller of allegro_debug_gemm that passes a NEW matrix calls allegro_debug_forget_weights first (it drops every cached packed
 * weight and tensor map of the handle; they are rebuilt on demand). */
int allegro_debug_set_precision(void* h, int passes);
int allegro_debug_forget_weights(void* h);
/* Test hook: capacity of the next list builds = E + frac * E + extra (default 0.125, 4096); (0, 0) forces the recovery path. */
int allegro_debug_set_list_slack(void* h, double frac, int64_t extra);
int allegro_debug_gemm(void* h, int64_t M, int64_t rows_cap, const float* A0, int lda0, int K0, const float* A1, int lda1, int K1,
                       const float* W, int ldw, int wtrans, int N, int pro, int epi, const float* aux, int ldaux, const float* geo,
                       float* C, int ldc, float* C2, int ldc2, int split, float c_old, float c_new, void* stream);

const char* allegro_last_error(void* h);

#ifdef __cplusplus
}
#endif
#endif /* ALLEGRO_B200_H */
