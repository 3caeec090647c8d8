/*
 * dmrg_b200.h — C ABI of the B200-native two-site DMRG effective-Hamiltonian library.
 *
 * The calls follow the problem statement of arxiv 2501.18263 (cited as PAPER.md:<line>):
 *   - the quantum-chemistry Hamiltonian, Eq. (1), with the 1/2 in front of
 *     the two-body sum (reading R1):
 *       H = sum_{ij,s} T_ij a+_{is} a_{js} + 1/2 sum_{ijkl,s,t} V_ijkl a+_{is} a+_{jt} a_{lt} a_{ks} + e_core
 *   - the MPS of PAPER.md Eq. (4) with U(1)xU(1) block-sparse tensors
 *   - the two-site effective space H_L (x) H_k (x) H_{k+1} (x) H_R
 *   - H_eff.psi as the task list of PAPER.md Eq. (6)-(8)
 *   - the "iterative eigensolver" of PAPER.md:63 (Davidson, DESIGN.md App. E)
 *   - the "renormalization steps" of PAPER.md:99 (operator blocking with an MPS tensor).
 *
 * Conventions:
 *   orbitals i = 0..L-1 along the chain; sites are 1-based in the API (site i = orbital i-1);
 *   site state s = 0..3 = {empty, down, up, up+down}, quantum numbers q(s) = (n_up, n_dn)
 *   = (0,0),(0,1),(1,0),(1,1), |3> = a+_up a+_dn |0>;
 *   bond b = 0..L lies between site b and b+1; a bond sector label q = (n_up, n_dn) counts the
 *   electrons in sites 1..b.  All matrices are row-major doubles.
 *
 * Memory and errors:
 *   Every function returns 0 on success and a negative dmrg_status on failure; the message of the
 *   last failure on a context is dmrg_last_error(ctx).  No exception crosses the boundary and there
 *   is no global state.  Pointers named h_* are HOST pointers (caller-owned, copied on entry or
 *   filled on return); pointers named d_* are DEVICE pointers on the context's device.  Device
 *   memory is obtained only through the allocator callbacks given at creation (the Python binding
 *   backs them with torch tensors); `stream` arguments are a cudaStream_t passed as void* and all
 *   device work of a call is enqueued on it.  Calls that return host results synchronise `stream`
 *   before returning; dmrg_heff_apply and dmrg_heff_diag do not synchronise.
 *   There is no CPU fallback: every numerical step runs in the library's CUDA kernels.
 */
#ifndef DMRG_B200_H
#define DMRG_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  DMRG_OK = 0,
  DMRG_ERR_ARG = -1,      /* invalid argument or call order */
  DMRG_ERR_INPUT = -2,    /* input violates a stated requirement (symmetry, isometry, shapes) */
  DMRG_ERR_ALLOC = -3,    /* allocator callback returned NULL */
  DMRG_ERR_CUDA = -4,     /* CUDA runtime error (message holds cudaGetErrorString) */
  DMRG_ERR_UNSUPPORTED = -5
} dmrg_status;

typedef struct dmrg_ctx dmrg_ctx;

/* Device allocator callbacks.  alloc returns a device pointer aligned to >= 256 bytes or NULL. */
typedef void* (*dmrg_alloc_fn)(uint64_t bytes, void* user);
typedef void (*dmrg_free_fn)(void* ptr, void* user);

typedef struct {
  int32_t L;            /* number of spatial orbitals ("d") */
  int32_t n_up, n_dn;   /* target electron numbers (N_alpha, N_beta); S_z = (n_up - n_dn)/2 */
  int32_t symmetry;     /* 0 = U(1)xU(1); 1 = SU(2) spin-adapted, total spin 0
                           only (n_up == n_dn): bond sectors are then labelled (N, 2S) in the q_up/q_dn arrays */
  int32_t device;       /* CUDA device ordinal */
  uint64_t workspace_bytes; /* cap for the intermediate (O_L.psi) buffer; 0 = library default */
  uint64_t env_cache_bytes; /* device cap for cached environment blocks (sweeps re-use them); 0 = 1/8 of device memory.
                               Over the cap the cached block farthest from the current bond is moved to the host tier
                               (env_host_bytes) or dropped; the two blocks in use do not count as removable */
  dmrg_alloc_fn alloc;
  dmrg_free_fn free;
  void* alloc_user;
  uint64_t env_host_bytes;  /* host tier of the environment cache: cached blocks that no longer fit the device cap are
                               moved to pinned host memory (up to this many bytes) instead of being dropped, and copied
                               back when a sweep needs them; 0 = no host tier */
} dmrg_config;

int dmrg_create(const dmrg_config* cfg, dmrg_ctx** out);
int dmrg_destroy(dmrg_ctx* ctx);
const char* dmrg_last_error(const dmrg_ctx* ctx);

/* PAPER.md Eq. (1).  h_T: L*L, h_V: L^4 with V[((i*L+j)*L+k)*L+l] the coefficient of
 * 1/2 a+_{is} a+_{jt} a_{lt} a_{ks}.  Requires T symmetric and V_ijkl = V_klij to 1e-12 (else
 * DMRG_ERR_INPUT).  The library uses w_ijkl = (V_ijkl + V_jilk)/2. */
int dmrg_load_integrals(dmrg_ctx* ctx, int32_t L, const double* h_T, const double* h_V, double e_core);

/* Bond sectors of the MPS (Eq. (4), :107).  For bond b = 0..L, sectors
 * sec_off[b] .. sec_off[b+1]-1 of the arrays (q_up, q_dn, dim), sorted lexicographically by
 * (q_up, q_dn) inside a bond.  Bond 0 must be {(0,0):1}, bond L {(n_up,n_dn):1}. */
int dmrg_mps_set_sectors(dmrg_ctx* ctx, const int32_t* h_sec_off /* L+2 */, const int32_t* h_q_up,
                         const int32_t* h_q_dn, const int32_t* h_dim);

/* Site tensor of site i (1-based).  Blocks are listed as (q_in index within bond i-1, site state s);
 * block n is the d_in x d_out matrix at h_data + blk_off[n], q_out = q_in + q(s) must be a sector of
 * bond i.  canonical = 0: left-canonical (sum_{q_in,s} A^T A = 1 on each q_out), 1: right-canonical
 * (sum_{s,q_out} A A^T = 1 on each q_in); violated beyond 1e-10 -> DMRG_ERR_INPUT. */
int dmrg_mps_set_site(dmrg_ctx* ctx, int32_t site, int32_t canonical, int32_t nblocks,
                      const int32_t* h_qin_idx, const int32_t* h_s, const int64_t* h_blk_off,
                      const double* h_data, void* stream);

/* SU(2) contexts: reduced site tensor of site i.  Block n maps (sector qin_idx[n] of bond
 * i-1, site multiplet m[n] = 0,1,2 = (N=0,S=0),(N=1,S=1/2),(N=2,S=0)) to sector qout_idx[n] of bond i, which must be
 * a spin coupling of the two; d_in x d_out row-major, counted in multiplets.  Coupling order:
 * left-canonical states |(block, site) S'>, right-canonical states |(site, block) S'>; a bond label (N, 2S) is the
 * content of sites 1..b, the right block of that bond carries (N_tot - N, S).  Isometry conditions as above. */
int dmrg_mps_set_site_su2(dmrg_ctx* ctx, int32_t site, int32_t canonical, int32_t nblocks,
                          const int32_t* h_qin_idx, const int32_t* h_m, const int32_t* h_qout_idx,
                          const int64_t* h_blk_off, const double* h_data, void* stream);

/* Replace the sectors of bond b (1 <= b <= L-1), e.g. after the SVD truncation of a sweep step changed the
 * kept states.  Arrays as in dmrg_mps_set_sectors for that one bond (sorted).  The site tensors of sites b
 * and b+1 and every cached environment that contains bond b become unset and must be given again. */
int dmrg_mps_update_bond(dmrg_ctx* ctx, int32_t b, int32_t nsec, const int32_t* h_q_up, const int32_t* h_q_dn,
                         const int32_t* h_dim);

/* Build the left environment from sites 1..k-1 and the right one from sites k+2..L by exact operator
 * blocking, then prepare the two-site problem at bond (k, k+1): complementary
 * operators, the task list of PAPER.md Eq. (8), and the diagonal of H_eff. */
int dmrg_env_build(dmrg_ctx* ctx, int32_t k, void* stream);

/* One renormalisation step: absorb site k into the left block (direction = 0, the
 * left-canonical tensor of site k must have been set) or site k+1 into the right block
 * (direction = 1), and prepare the two-site problem at the shifted bond (k+1,k+2) or (k-1,k).
 * The environment on the other side comes from the environment cache (blocks built earlier for the same site
 * tensors) or is rebuilt from the stored site tensors. */
int dmrg_renormalize(dmrg_ctx* ctx, int32_t direction, void* stream);

/* Layout of the two-site wavefunction Psi_{a, s_k, s_{k+1}, b}: blocks ordered by
 * (q_L lexicographic, s_k, s_{k+1}); block n is a d_L x d_R row-major matrix at offset off[n] of the
 * flat vector.  Pass NULL arrays to query only *nblocks / *n.
 * SU(2) contexts: reduced blocks of |((a, m1) S', (m2, b) S') S_tot = 0>, ordered by (q_L, m1, S' ascending, m2,
 * q_R ascending in S); qL_up/qL_dn = (N, 2S) of bond k-1, s1/s2 = multiplets m1/m2, qR_up/qR_dn = (N, 2S) label of
 * bond k+1, twoS_mid = 2S'. */
typedef struct {
  int32_t qL_up, qL_dn;   /* label of bond k-1 */
  int32_t s1, s2;         /* site states of sites k, k+1 */
  int32_t qR_up, qR_dn;   /* label of bond k+1 (electrons in sites 1..k+1) */
  int32_t dL, dR;
  int64_t off;
  int32_t twoS_mid;       /* SU(2) only: doubled spin S' of L' = L + site k (= spin of R'), else 0 */
  int32_t pad_;
} dmrg_psi_block;
int dmrg_psi_layout(dmrg_ctx* ctx, int32_t* nblocks, dmrg_psi_block* h_blocks, int64_t* n);

/* psi_out = H_eff psi_in (Eq. (7)/(8)); e_core is included.  Overwrites d_psi_out. */
int dmrg_heff_apply(dmrg_ctx* ctx, const double* d_psi_in, double* d_psi_out, void* stream);

/* Sharding of H_eff.psi over `count` ranks, one process per GPU (the tasks are "independent operations";
 * PAPER.md:25 multi-GPU).  Call before dmrg_env_build / dmrg_renormalize.  Every rank holds the whole MPS and both
 * environments and prepares the same two-site problem; the psi' blocks are dealt to the ranks by analytic flops
 * (largest first to the least loaded rank — the same map on every rank), and rank r keeps only the tasks whose
 * OUTPUT block it owns.  A psi' block is therefore computed completely by one rank and is exactly zero on the
 * others, so the exchange is a plain sum.  With `reduce` set, dmrg_heff_apply and dmrg_davidson call
 * reduce(user, d_buf, n, stream) after the local tasks of every apply; it must replace the n doubles at the device
 * pointer d_buf by their sum over all ranks, enqueued on `stream` (the binding uses torch.distributed.all_reduce over
 * NCCL), and return 0.  With reduce = NULL dmrg_heff_apply returns the rank's partial result (e_core.psi is added
 * by rank 0 only) and the caller sums; dmrg_davidson then fails with DMRG_ERR_ARG.  diag(H_eff) is whole on every
 * rank.  count = 1 restores the unsharded library. */
typedef int (*dmrg_reduce_fn)(void* user, double* d_buf, int64_t n, void* stream);
int dmrg_set_shard(dmrg_ctx* ctx, int32_t rank, int32_t count, dmrg_reduce_fn reduce, void* user);

/* Owner rank of every psi block (h_owner: nblocks ints) and the analytic flops per rank (h_flops: `count` doubles)
 * of the prepared problem; either pointer may be NULL. */
int dmrg_shard_info(dmrg_ctx* ctx, int32_t* h_owner, double* h_flops);

/* Analytic flops of one H_eff.psi per OUTPUT block of psi' (sum over the tasks that write the block of
 * the cheaper contraction order on the unpadded dims); h_flops: nblocks doubles, their sum is dmrg_stats.flops_apply
 * of an unsharded context.  Used to quote the CPU oracle's rate on a sample of blocks in the same flop count. */
int dmrg_block_flops(dmrg_ctx* ctx, double* h_flops);

/* Diagonal of H_eff in the psi layout. */
int dmrg_heff_diag(dmrg_ctx* ctx, double* d_diag, void* stream);

/* Davidson for the lowest eigenpair (DESIGN.md App. E).  d_psi holds the start vector on entry and
 * the normalised Ritz vector on return.  *iters = number of H_eff applications. */
int dmrg_davidson(dmrg_ctx* ctx, double* d_psi, double tol, int32_t max_iter, int32_t max_basis,
                  double* h_energy, int32_t* h_iters, double* h_resid, void* stream);

/* Convenience end-to-end variants with HOST vectors (copies inside the call). */
int dmrg_heff_apply_host(dmrg_ctx* ctx, const double* h_psi_in, double* h_psi_out, void* stream);
int dmrg_davidson_host(dmrg_ctx* ctx, double* h_psi, double tol, int32_t max_iter, int32_t max_basis,
                       double* h_energy, int32_t* h_iters, double* h_resid, void* stream);

/* ---- mode-optimisation micro-iteration (Sec. II.B, :57-75, Fig. 1 :63), steps ii) and iii); U(1)xU(1) ----
 *
 * dmrg_two_site_gate: psi_out{a, s1' s2', b} = sum_{s1 s2} G[(s1' s2'), (s1 s2)] psi_in{a, s1 s2, b} for a 16 x 16
 * row-major gate h_G on the occupation basis of sites k, k+1 (index 4 s1 + s2).  G must conserve (n_up, n_dn) of the
 * pair (DMRG_ERR_INPUT otherwise).  For the orbital rotation c~+_k = cos(theta) c+_k + sin(theta) c+_{k+1},
 * c~+_{k+1} = -sin(theta) c+_k + cos(theta) c+_{k+1} (both spins), the coefficients of the same state in the rotated
 * modes are G = exp(-theta kappa) psi with kappa = sum_s (c+_{k+1,s} c_{k,s} - c+_{k,s} c_{k+1,s}); theta = pi/2 is the
 * swap gate of PAPER.md:89 up to signs.  d_psi_in and d_psi_out must not alias.  Synchronises `stream`.
 *
 * dmrg_bond_entropy: block entropies of rho_{1..k} (the cut between the two sites) of the two-site wavefunction
 * d_psi: *h_S_half = S_1/2 = 2 ln Tr sqrt(rho) (the cost function of PAPER.md:75), *h_S_vn = -Tr rho ln rho; psi is
 * normalised internally.  The singular values of Psi[(a s_k), (s_{k+1} b)] are computed per sector of bond k by a
 * one-sided Jacobi kernel in shared memory (DMRG_ERR_UNSUPPORTED if a sector exceeds ~160 x 160: the paper runs mode
 * optimisation at D <= 256); h_sigma (optional, host) receives them unnormalised, sector by sector
 * (sectors of bond k in lexicographic order), *n_sigma their number.  Any output pointer may be NULL.
 *
 * dmrg_rotate_integrals: T and V are replaced by the integrals in the rotated modes (k, k+1 1-based sites,
 * same theta convention), so that H is unchanged as an operator; all environments become invalid
 * (call dmrg_env_build again).  Host work only. */
int dmrg_two_site_gate(dmrg_ctx* ctx, const double* h_G, const double* d_psi_in, double* d_psi_out, void* stream);
/* h_G (16 x 16, row-major) = exp(-theta kappa), the gate of the orbital rotation described above (host). */
int dmrg_rotation_gate(double theta, double* h_G);
int dmrg_bond_entropy(dmrg_ctx* ctx, const double* d_psi, double* h_S_half, double* h_S_vn, double* h_sigma,
                      int32_t* n_sigma, void* stream);
int dmrg_rotate_integrals(dmrg_ctx* ctx, int32_t k, double theta);

/* dmrg_bond_entropy_static: dmrg_bond_entropy (same arguments, same kernels, same results) for callers that may not
 * allocate device memory: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  It
 * calls no cudaMalloc / cudaFree, none of the context's allocator callbacks and no allocating library routine: the
 * sector tables, the singular values and the three results live in one file-scope `static __device__` array of
 * ~124 KiB, which every GPU that loads the library holds until the process exits.  Its device address is looked up
 * once per device (cudaGetSymbolAddress, on the first call with a context of that device).
 *   Limits (DMRG_ERR_UNSUPPORTED beyond them, with the count in dmrg_last_error; dmrg_bond_entropy has none of them):
 * at most DMRG_STATIC_MAX_SIGMA singular values (sum over the sectors of bond k of min(rows, columns): enough for
 * D <= 512), DMRG_STATIC_MAX_SECTORS sectors of bond k and DMRG_STATIC_MAX_BLOCKS psi blocks.
 *   d_psi: device, read only.  h_*: host, optional as in dmrg_bond_entropy.  Synchronises `stream`.
 *   ALL calls in the process that use one GPU share the array, across contexts and threads: calls that overlap on the
 * GPU (two streams, two host threads) race and return garbage; serialise them.  The array keeps the last call's
 * contents; every word a kernel reads is written earlier in the same call and the result slot is cleared first. */
#define DMRG_STATIC_MAX_SIGMA 2048
#define DMRG_STATIC_MAX_SECTORS 512
#define DMRG_STATIC_MAX_BLOCKS 4096
int dmrg_bond_entropy_static(dmrg_ctx* ctx, const double* d_psi, double* h_S_half, double* h_S_vn, double* h_sigma,
                             int32_t* n_sigma, void* stream);

/* ---- truncation step of a micro-iteration ("keeping only the D largest singular values in SVD"; Fig. 1
 * :63 "SVD"; the "SVD" and "StVec" columns of the paper's timing table :284); U(1)xU(1) ----
 *
 * dmrg_truncate_bond: d_psi (device, read only) is the optimised two-site wavefunction of the prepared problem at bond
 * (k, k+1).  Psi[(a s_k), (s_{k+1} b)] is decomposed per sector of bond k by a one-sided Jacobi SVD on the device;
 * the D largest singular values over all sectors are kept (values <= 1e-14 never; equal values: the sector that comes
 * first in lexicographic (n_up, n_dn) order first, R23).  The library then replaces its sectors of bond k by
 * the kept ones and installs, without a host round trip, the new left-canonical tensor of site k (direction 0, the
 * sweep moves right: A = U) or the new right-canonical tensor of site k+1 (direction 1: B = V^T); the tensor of the
 * other centre site becomes unset and cached environment blocks that contain either site are dropped, exactly as
 * dmrg_mps_update_bond + dmrg_mps_set_site would do.  The prepared problem stays prepared: call
 * dmrg_renormalize(direction) next.  *h_discarded = sum of the squares of the singular values not among the D largest;
 * *h_kept = number of kept states (both host, optional).
 *   The Jacobi kernel holds a sector matrix in the shared memory of one CTA when rows x columns <= ~27 000 (~165 x 165:
 * bond dimensions up to D ~ 256, the regime of the paper's mode optimisation); a larger sector is rotated in place in
 * global memory, which is correct at any size but slow (a caller at large D may prefer its own SVD with
 * dmrg_mps_update_bond / dmrg_mps_set_site).  DMRG_ERR_UNSUPPORTED for SU(2) contexts (nothing changed then).
 * Synchronises `stream`.
 *
 * dmrg_start_vector: after dmrg_truncate_bond(direction) and dmrg_renormalize(direction), d_psi_out (device,
 * dmrg_psi_layout of the NEW problem) receives the wave-function transformation of the truncated state: the centre
 * factor Sigma V^T (or U Sigma) contracted with the canonical tensor of the site that joined the two-site centre.  Not
 * normalised.  DMRG_ERR_ARG if the calls did not come in that order.  Synchronises `stream`.
 *
 * dmrg_bond_sectors: the sectors of bond b (0..L) as the library holds them, in lexicographic order; *nsec always,
 * the arrays (host, capacity >= *nsec, any may be NULL) when given. */
int dmrg_truncate_bond(dmrg_ctx* ctx, const double* d_psi, int32_t direction, int32_t D, double* h_discarded,
                       int32_t* h_kept, void* stream);
int dmrg_start_vector(dmrg_ctx* ctx, double* d_psi_out, void* stream);
int dmrg_bond_sectors(dmrg_ctx* ctx, int32_t b, int32_t* nsec, int32_t* h_q_up, int32_t* h_q_dn, int32_t* h_dim);

typedef struct {
  int64_t n_terms;          /* four-part terms of PAPER.md Eq. (6) after pre-summation */
  int64_t n_tasks;          /* (term x sector) tasks of PAPER.md Eq. (8) */
  int64_t n_groups;         /* batched task groups handed to the kernel */
  double flops_apply;       /* analytic: sum over tasks of the cheaper contraction order */
  double flops_executed;    /* flops the kernels issue for one apply (padding included) */
  double bytes_unique;      /* operator blocks once + psi in/out */
  double bytes_intermediate;/* O_L.psi intermediates written+read per apply */
  int64_t psi_size;         /* length of the flat psi vector */
  int64_t op_bytes_left, op_bytes_right;
  int32_t n_chunks;         /* workspace chunks per apply */
  int32_t launches_per_apply;
  double last_build_ms;     /* host+device time of the last dmrg_env_build / dmrg_renormalize */
  double flops_renorm;      /* analytic flops of the last renormalisation step */
  int64_t total_launches;   /* kernels launched by this context so far */
  double renorm_ms;         /* host+device time of the single blocking step of the last dmrg_renormalize */
  double flops_shared;      /* phase-1 flops per apply saved by sharing O_L.psi intermediates between term groups */
  int64_t env_spills, env_fetches;   /* environment blocks moved to / back from the host tier so far */
  double env_host_bytes;    /* pinned host memory held by the host tier */
  double env_device_bytes;  /* device-resident bytes of the cached environment blocks */
} dmrg_stats_t;
int dmrg_stats(dmrg_ctx* ctx, dmrg_stats_t* out);

/* Export one carried block operator (for parity tests).  side 0 = left, 1 = right.  kind:
 * 0 H, 1 C_up, 2 C_dn, 3 A_upup, 4 A_updn, 5 A_dndn, 6 B_upup, 7 B_updn, 8 B_dndn, 9 S_up, 10 S_dn.
 * (i, j) are orbital indices (j ignored for one-index kinds).  The operator is returned as a dense
 * (D x D) row-major matrix over the block's states in sector order, D = sum of sector dims.
 * Right-block sectors are ordered by their bond label (electrons LEFT of the bond). */
int dmrg_env_export(dmrg_ctx* ctx, int32_t side, int32_t kind, int32_t i, int32_t j,
                    double* h_out, int64_t* D);

/* One sector block of EVERY operator of a carried class (parity tests at sizes where the dense matrices of
 * dmrg_env_export are too large: BASELINE configs 3 and 4).  U(1)xU(1) contexts: `kind` as in dmrg_env_export and
 * `d2S` is ignored.  SU(2) contexts: kind 0 H, 1 C (rank 1/2), 2 A^0, 3 A^1, 4 B^0, 5 B^1, 6 S~ (rank 1/2) — the reduced
 * elements X_red[S',S] of <S'M'|X^k_q|SM> = <S M; k q|S' M'> X_red[S',S] — and d2S = 2S' - 2S selects the
 * class.  side: 0 / 1 = the left / right block of the prepared problem; 2 = the cached left block of sites 1..k-2,
 * 3 = the cached right block of sites k+3..L (the predecessors of one blocking step; DMRG_ERR_ARG if the
 * environment cache no longer holds them on the device).  The block is chosen by the label of its INPUT sector, (q_up, q_dn) resp. (N, 2S), in the convention of
 * dmrg_psi_block: left block = content of the block, right block = label of the bond (electrons LEFT of it).
 * Returns *nops, *rows (output sector), *cols (input sector) and, if h_out != NULL, the nops x rows x cols
 * row-major array; *rows = *cols = 0 if the class has no block with that input sector.  Operator order inside a
 * class: C, S: orbitals ascending (S: the orbitals OUTSIDE the block); A_upup, A_dndn, A^1: pairs i < j, i-major;
 * A^0: pairs i <= j, i-major; A_updn, B_*, B^0, B^1: (i, j) row-major over the block's orbitals. */
int dmrg_env_export_block(dmrg_ctx* ctx, int32_t side, int32_t kind, int32_t d2S, int32_t qin_a, int32_t qin_b,
                          int32_t* nops, int32_t* rows, int32_t* cols, double* h_out);

/* The factor F of PAPER.md Eq. (10)-(11) (host; doubled-spin arguments): *h_F_ninej = the rescaled Wigner 9j
 * closed form sqrt((2Sa'+1)(2Sk'+1)(2Sg+1)(2k+1)) {Sa Sk Sg; kL kk k; Sa' Sk' Sg'}, *h_F_contraction = the contraction
 * of six Clebsch-Gordan tensors of PAPER.md Fig. 4 from the library's own CG table (the table all SU(2) task
 * prefactors are built from). */
int dmrg_su2_f_factor(int32_t twoSa, int32_t twoSk, int32_t twoSg, int32_t twokL, int32_t twokk, int32_t twok,
               int32_t twoSa_out, int32_t twoSk_out, int32_t twoSg_out, double* h_F_ninej, double* h_F_contraction);

/* Measured FP64 tensor-pipe (DMMA) peak of the device in TFLOP/s: a register-only mma loop on all
 * SMs, timed with CUDA events on `stream`. */
int dmrg_fp64_peak(dmrg_ctx* ctx, double* h_tflops, void* stream);
/* The same measurement with plain DFMA instructions (FP64 vector pipe) instead of DMMA: the second comparison peak of
 * SURVEY.md 8(d). */
int dmrg_dfma_peak(dmrg_ctx* ctx, double* h_tflops, void* stream);

/* Per-launch timing of one H_eff.psi (measurement aid): runs dmrg_heff_apply with every
 * kernel launch of the task plan bracketed by CUDA events on `stream` and synchronises.  Up to `cap`
 * records are written to h_out; *n receives the number of launches.  phase 1 = O_L.psi (or psi.O_R^T)
 * into the workspace, phase 2 = accumulation into psi'; shape = tile shape index 3*row_class+col_class
 * with classes {32,64,128}, -1 = split-K reduction; flops = flops the launch's tiles execute. */
typedef struct {
  int32_t chunk, phase, shape, ntiles;
  double flops;
  double ms;
} dmrg_launch_info;
int dmrg_apply_profile(dmrg_ctx* ctx, const double* d_psi_in, double* d_psi_out, int32_t cap,
                       dmrg_launch_info* h_out, int32_t* n, void* stream);

#ifdef __cplusplus
}
#endif
#endif
