/*
 * p3t.h -- C ABI of the B200-native soft-force library for the P3T scheme
 *          (arXiv 1506.04553, Iwasawa, Portegies Zwart, Makino).
 *
 * What the library computes (citations: PAPER.md line, equation):
 *   for every particle i, on one GPU (L138, L142-153 steps 1 and 7),
 *     a_i   = - sum_{j != i} m_j K(s_ij) (q_i - q_j) / s_ij^3      (Eq. 8, per unit mass)
 *     phi_i = - sum_{j != i} m_j W(s_ij) / s_ij                     (Eq. 6, per unit mass)
 *     L_i   = { j != i : s_ij < r_search }                          (L138-140, h = r_cut + dr_buff)
 *   with s_ij = sqrt(|q_i - q_j|^2 + eps^2) (Eq. 2), K the cutoff function of
 *   Eq. 12 (L85), W the transition function of Eq. 16-17 (L102-104), G = 1 (L163),
 *   by a Barnes-Hut octree with monopole + quadrupole cells (L138) opened with the
 *   parameter theta (L171, L193).  r_out is the paper's r_cut, r_search its h.
 *
 * All arithmetic runs in hand-written sm_100a CUDA kernels; there is no CPU
 * fallback.  Pair and cell interactions are evaluated in fp32; every 128
 * interactions the fp32 partial sums are added to fp64 accumulators.
 *
 * Conventions
 *   - Pointers marked [device] must be device memory of the context's GPU,
 *     [host] host memory; calls with an `on_device` flag accept either.
 *   - Ownership: the caller owns every buffer it passes, including the
 *     workspace; the library copies inputs into the workspace and never frees
 *     caller memory.  The p3t_ctx itself is host heap, freed by p3t_destroy.
 *   - Errors: every call returns a p3t_status; nothing aborts or throws.
 *     p3t_last_error() gives a message for the last failing call on that ctx.
 *   - Asynchrony: load/build/eval only enqueue work on the context's stream.
 *     Calls that write host memory synchronise the stream before returning.
 *   - Thread safety: one thread per context at a time.
 */
#ifndef P3T_H
#define P3T_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct p3t_ctx p3t_ctx;

typedef enum {
    P3T_OK        =  0,
    P3T_EINVAL    = -1,  /* bad argument: n = 0, n > max_n, non-finite input, eps < 0, theta < 0,
                            not (0 <= r_in < r_out <= r_search), unknown enum value, null pointer */
    P3T_ESTATE    = -2,  /* call order: build before load, eval before build, fetch before eval */
    P3T_ENOMEM    = -3,  /* workspace too small, or host allocation failed */
    P3T_ECAPACITY = -4,  /* neighbour buffer (nbr_capacity) or a caller's output buffer too small;
                            the true total is still reported by p3t_get_neighbour_counts */
    P3T_ECUDA     = -5,  /* a CUDA runtime call failed; see p3t_last_error */
    P3T_ELIMIT    = -6   /* the Hermite part needed more than max_blocks block steps */
} p3t_status;

/* Per-call statistics.  Interaction counts are pair evaluations for real
 * particles (padded lanes of partly filled groups are not counted); the flop
 * convention of DESIGN.md (23 per p-p, 65 per p-c) is applied by the caller. */
typedef struct {
    uint64_t n;              /* particles loaded */
    uint64_t n_pp;           /* particle-particle interactions of the last eval */
    uint64_t n_pc;           /* particle-cell (monopole+quadrupole) interactions */
    uint64_t n_near;         /* of n_pp: pairs evaluated on the K/W + neighbour-test path */
    uint64_t n_neighbours;   /* sum of list lengths (ordered pairs) of the last eval */
    uint32_t n_cells;        /* octree cells (internal + leaf) */
    uint32_t n_leaves;
    uint32_t n_groups;       /* i-groups walked (one warp each) */
    uint32_t depth;          /* deepest level in use (root = 0) */
    uint32_t max_list;       /* longest neighbour list */
    uint32_t sort_passes;    /* radix passes of the last build (8-bit digits; at most 8 for 63-bit keys, 4 for 30-bit keys: p3t_set_sort_passes) */
    float ms_sort;           /* a1-a4: bounding cube, keys, radix sort, gather */
    float ms_build;          /* a5: octree + groups */
    float ms_moments;        /* a6 */
    float ms_walk;           /* a7-a8 */
    float ms_nbr;            /* a9 */
    float ms_hard;           /* last p3t_eval_hard */
    float ms_pack;           /* a1: pack + bounding cube of the last p3t_load_particles (after any host-to-device copy) */
    uint32_t tree_refits;    /* p3t_refit_tree: refits since the last full build (0: the current tree is a fresh build) */
    uint32_t n_stray;        /* of the current refit: bodies outside the cube of their leaf by more than stray_dist leaf sides */
    uint32_t walk_parts;     /* how the last walk mapped groups to warps: 1 one warp per group, 2 / 4 split walk, 0 one CTA per group */
    uint32_t sort_max_run;   /* last build, if it sorted the upper key bits only: longest run of keys equal on them that the
                                finishing step had to sort, 0 if none was longer than 16 */
} p3t_stats;

/* Bytes of device workspace p3t_create needs for up to max_n particles,
 * key_bits in {30, 63} and room for nbr_capacity neighbour entries (ordered
 * pairs, summed over all lists).  Returns 0 for invalid arguments. */
size_t p3t_workspace_bytes(size_t max_n, int key_bits, size_t nbr_capacity);

/* Create a context on `device` working on `cuda_stream` (a cudaStream_t passed
 * as void*; NULL = the legacy default stream).  `workspace` [device] must be
 * 256-byte aligned, at least p3t_workspace_bytes(...) long and stay alive until
 * p3t_destroy.  Defaults: nleaf = 16, ngroup = 64; parameters must be set with
 * p3t_set_params before the first build. */
p3t_status p3t_create(p3t_ctx **out, int device, size_t max_n, int key_bits,
                      void *workspace, size_t workspace_bytes, size_t nbr_capacity, void *cuda_stream);
p3t_status p3t_destroy(p3t_ctx *ctx);

/* eps: Plummer softening (Eq. 2); theta: opening parameter, 0 = open every
 * cell (the tree path then is the direct sum); r_in, r_out: inner and outer
 * cutoff radii of K and W (Eq. 12-17; r_out = r_cut); r_search: neighbour
 * radius h >= r_out (L138-140).  Changing them invalidates a built tree
 * (theta and r_search enter the per-cell acceptance radius). */
p3t_status p3t_set_params(p3t_ctx *ctx, float eps, float theta, float r_in, float r_out, float r_search);

/* Per-pair-class cutoffs (section 3.2.2.1: "We use three values for the cut off
 * radius with respect to three different kinds of interactions").  cls[n] gives every particle (user order) a class,
 * 0 = field star (FS), 1 = black hole (BH); the kind of a pair is class_i + class_j:
 *   0  FS-FS  r_in, r_out, r_search, eps of p3t_set_params                       (paper: r_cut,FS-FS = 1/256)
 *   1  BH-FS  r_in_bf, r_out_bf, r_search_bf, the same eps                        (paper: r_cut,BH-FS = 1/32)
 *   2  BH-BH  not split: "the force is not split and F_soft = 0 ... integrated with the pure Hermite scheme": K = W = 0
 *             in a_i and phi_i at every separation, the two are ALWAYS in each other's list, and the hard part
 *             (p3t_eval_hard) gives them the whole Newtonian term with the softening eps_bb (paper: none)
 * in every formula of this header (Eq. 6-8, the list rule).  A cell is used as a multipole only if every body in it is a
 * plain Newtonian partner of every body of the group: a cell or a group that holds a black hole keeps clear of
 * max(r_search, r_search_bf), and a group with a black hole opens every cell that holds one.  The split kinds share
 * one softening, as in the paper's runs, because a cell term has only one.
 * cls is host or device memory (on_device); it is copied, the classes stay with the particle ids over later
 * p3t_load_particles calls of the same n.  cls = NULL switches classes off.  A built tree becomes invalid.
 * P3T_EINVAL: n = 0 or > max_n, a class above 1 (host input; device input is reduced to its lowest bit), not
 * (0 <= r_in_bf < r_out_bf <= r_search_bf), eps_bb < 0, non-finite values.  P3T_ESTATE from p3t_build_tree and
 * p3t_eval_direct when n differs from the loaded particle count.  p3t_hermite_step and p3t_step integrate with the
 * kind's own force too (two black holes: the pure Hermite scheme, unsoftened by default); the accuracy parameters of
 * class 1 come from p3t_set_hermite_class_params (L287: eta_FS = 0.1, eta_BH = 0.03). */
p3t_status p3t_set_pair_classes(p3t_ctx *ctx, size_t n, const uint8_t *cls, int on_device, float r_in_bf, float r_out_bf,
                                float r_search_bf, float eps_bb);

/* nleaf in 1..32: a cell with more than nleaf bodies is split (unless at the
 * key depth limit); ngroup in {32, 64}: bodies per i-group (one warp). */
p3t_status p3t_set_tree_params(p3t_ctx *ctx, int nleaf, int ngroup);

/* Space-filling curve of the keys (row a2).  0: Morton (bit-interleaved quantised coordinates, what north_star names);
 * 1 (default): Peano-Hilbert -- the same quantised coordinates taken through Skilling's transform before the
 * interleave.  Both give the same octree (a level-l cell is the run of keys sharing their top 3 l bits; only the order
 * of the octants inside a cell differs), the same cells, moments and, up to the grouping of the targets, the same
 * results; the Hilbert order makes consecutive bodies neighbours in space everywhere, so i-groups can be plain runs of
 * ngroup consecutive bodies with full warps and tight boxes (A25, section 7).  Invalidates a built tree.
 * P3T_EINVAL for another value. */
p3t_status p3t_set_key_curve(p3t_ctx *ctx, int curve);

/* Radix passes of the sort (row a3).  The result of a build is always the stable order of the full keys.  passes = 0
 * (default): the library sorts only the upper digits by radix passes -- as many bits as the tree is expected to be deep,
 * log2 n + 14, eight more after every build whose statistics (read at the next synchronising call) show a run above 24
 * keys -- and finishes the runs of keys that agree on those bits in place (insertion sort by one thread up to 32 keys,
 * one CTA per longer run): the same permutation with 4 or 5 passes instead of 8 for the workloads of BASELINE.json.
 * passes = 1..8: that many of the upper digits by radix passes (8 with 63-bit keys, 4 or more with 30-bit keys: all of
 * them, no finishing step).  30-bit keys always take their 4 passes by default.  Invalidates a built tree.
 * P3T_EINVAL for a value outside 0..8. */
p3t_status p3t_set_sort_passes(p3t_ctx *ctx, int passes);

/* Inspection (host only, no GPU involved): the state tables the key kernel uses for Peano-Hilbert keys, derived by the
 * library from Skilling's transform on a 32^3 lattice.  tab[state * 64 + two octants] = next state << 6 | two key digits
 * (24 states, the root cell has state 0; an octant is 4 x-bit + 2 y-bit + z-bit), then tab[1536 + state * 8 + octant] =
 * next state << 3 | key digit.  words >= 1728.  P3T_EINVAL for bad arguments, P3T_ECUDA if the derivation found the
 * curve not to be a state machine (cannot happen; the same test guards p3t_create). */
p3t_status p3t_hilbert_state_tables(uint32_t *tab, size_t words);

/* Tuning: how many octree levels above its natural level (the level whose cell holds <= ngroup
 * bodies) an i-group's bodies may straddle.  0 = every group is one octree cell (partly filled
 * warps); 1 (default) = consecutive sibling cells are merged up to ngroup bodies.  Where the natural
 * level is above tree level 4 (sparse outskirts) groups never straddle, whatever this value.  Results
 * do not depend on it beyond rounding and the R-MAC box B. levels in 0..4, or 32: no cuts at all, every group is a plain
 * run of ngroup consecutive bodies (meant for the Peano-Hilbert order). */
p3t_status p3t_set_group_merge_levels(p3t_ctx *ctx, int levels);

/* How i-groups are mapped to warps in the tree walk.  1: one warp per group -- results are bitwise
 * reproducible.  2: the four warps of a CTA share one group through a common stack -- keeps the GPU busy
 * when there are few groups (small n) and shortens the tail of the launch; which warp evaluates which
 * cell depends on timing, so accelerations and potentials are reproducible to fp32 rounding of the
 * batch sums (a few 1e-6 relative at most) rather than bitwise; neighbour lists are identical.  3, 4: split walk -- 2 or 4
 * warps per group, each walking every 2nd / 4th cell of one tree level and everything below it, their sums added in a
 * fixed order by a small kernel (bitwise reproducible; sums differ from mode 1's by the rounding of the partial sums):
 * for mid-size n, where all groups start at once and the launch would end in a long tail of lone warps.  0 (default):
 * chosen from n / ngroup per resident warp (mode 2 below 0.3, mode 4 below 0.65, mode 3 below 1.3, else mode 1).
 * P3T_EINVAL for another value. */
p3t_status p3t_set_walk_mode(p3t_ctx *ctx, int mode);

/* Sharding of one evaluation over `world` GPUs: every rank loads ALL particles and builds the
 * same tree; p3t_eval_soft of the context with shard (rank, world) walks only the i-groups at positions rank,
 * rank + world, rank + 2 world, ... of the hand-out order.  Accelerations, potentials and neighbour lists of the
 * particles of the other groups come out as zero / empty, so the results of all ranks combine by addition of
 * acc and pot and concatenation of the lists (paper_1506_04553_b200/multi.py does it with torch.distributed).
 * Default (0, 1): everything.  P3T_EINVAL unless 0 <= rank < world. */
p3t_status p3t_set_shard(p3t_ctx *ctx, int rank, int world);

/* The exchange of a sharded evaluation as ONE all-reduce (sum) over the ranks.  p3t_get_shard_record writes, for every
 * particle in user order, five floats to rec[5n] [device]: (a_x, a_y, a_z, phi, cost class + 1) -- all zero for the
 * particles of the groups other ranks walked, so the sum over the ranks holds the acceleration, the potential and the
 * cost class of every particle.  p3t_put_shard_classes hands the summed record back [device]: the context takes the cost
 * classes from it, and since every rank now holds the same classes, the next p3t_eval_soft orders the groups by
 * predicted cost on every rank alike (an order kernel without atomics) and deals the positions of that order round
 * robin to the ranks -- each rank gets the same mix of expensive and cheap groups, longest first (SURVEY.md 8(e):
 * "balanced by the previous call's per-group interaction counts").  Without the exchange a sharded walk deals the groups
 * out in key order.  Both calls only enqueue.  P3T_ESTATE before an eval call; P3T_EINVAL for a null pointer.
 * (paper_1506_04553_b200/multi.py: allreduce_shard.) */
p3t_status p3t_get_shard_record(p3t_ctx *ctx, float *rec);
p3t_status p3t_put_shard_classes(p3t_ctx *ctx, const float *rec);

/* Load n particles: mass[n], pos[3n] (x,y,z interleaved), both host or both
 * device (on_device).  Every value is tested for being finite by the kernel that
 * packs the bodies.  Host data: the call waits for the copies and that kernel and
 * returns P3T_EINVAL itself (the host arrays may be reused when it returns); device
 * data: the call only enqueues, and the error surfaces at the next call that
 * synchronises. */
p3t_status p3t_load_particles(p3t_ctx *ctx, size_t n, const float *mass, const float *pos, int on_device);

/* a1-a6: bounding cube, Morton keys, radix sort, body gather, octree + groups,
 * moments (mass, centre of mass, quadrupole, acceptance radius). */
p3t_status p3t_build_tree(p3t_ctx *ctx);

/* Tree reuse between soft steps (PAPER.md L27-29 (section 1): "the cost of the usual complete
 * reconstruction of the tree is O(N log N) and not negligible"; the cost model counts one tree per soft step, L193 and
 * Eq. 28).  p3t_refit_tree replaces p3t_build_tree after a p3t_load_particles of the SAME particles (same n, same
 * order) at moved positions: sorted order, cells and i-groups of the last full build are kept; bodies are gathered again
 * and moments, tight boxes and acceptance radii are made from the new positions on the old topology (no keys, no sort,
 * no build).  Results keep the guarantees of a fresh tree -- accepted cells hold no body within r_search of the group
 * (lists exact), and the opening test uses, for a cell whose bodies have left its cube, the side of the smallest cube
 * about the cell's geometric centre that holds them -- what degrades is only how tight cells and groups are, i.e. the
 * number of interactions.  The call counts on the device the bodies that sit outside the cube of their leaf by more than
 * stray_dist leaf sides; if they are more than max_stray_fraction * n, or max_refits refits have been made since the
 * last build, or there is no tree to reuse (first call, n or tree parameters changed), the call does a full
 * p3t_build_tree instead.  It synchronises the stream once (to read the count).  p3t_set_params may change between refits.
 * Defaults: max_refits = 0 (p3t_refit_tree always rebuilds; p3t_step uses this call, so it rebuilds every step unless
 * reuse is switched on), stray_dist = 0.5, max_stray_fraction = 0.02.  P3T_EINVAL for negative or non-finite values. */
p3t_status p3t_set_tree_reuse(p3t_ctx *ctx, int max_refits, float stray_dist, float max_stray_fraction);
p3t_status p3t_refit_tree(p3t_ctx *ctx);

/* a7-a9: group walk, interactions, neighbour lists.  Needs a tree built for the
 * loaded positions and current parameters. */
p3t_status p3t_eval_soft(p3t_ctx *ctx);

/* Verification entry: brute-force O(N * n_subset) evaluation with the same K, W
 * and neighbour rule, no tree.  i_subset [same side as on_device] lists the
 * targets (user ids); NULL = all particles.  Results are fetched with the same
 * p3t_get_* calls; for a subset, entries of other particles are zero / empty. */
p3t_status p3t_eval_direct(p3t_ctx *ctx, const uint32_t *i_subset, size_t n_subset, int on_device);

/* The same brute-force evaluation for callers that cannot allocate device memory (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc): no context, no workspace.  For all n particles,
 *   acc[3 i ..] = - sum_{j != i} m_j K(s_ij) (q_i - q_j) / s_ij^3   (Eq. 8),   pot[i] = - sum_{j != i} m_j W(s_ij) / s_ij   (Eq. 6),
 *   nbr_count[i] = #{ j != i : s_ij < r_search }   (the list rule; nullable),
 * with the arithmetic of p3t_eval_direct (fp32 pair terms, one fp64 add per 128 sources).  mass [n], pos [3 n], acc
 * [3 n], pot [n], nbr_count [n] and info [2] (nullable: info[0] = sum of the counts, info[1] = number of non-finite
 * inputs, whose results are then meaningless) are DEVICE pointers on `device`, owned by the caller; cuda_stream is a
 * cudaStream_t (NULL = the legacy default stream).  Asynchronous on that stream.
 * Scratch (the bodies packed as float4 and a header of counters) is a file-scope device array of the library, sized for
 * P3T_STATIC_MAX_N particles: 1 MiB + 256 B that every GPU which loads the library holds until the process exits.  The
 * call makes no cudaMalloc / cudaFree and calls no allocating routine; its first call per device looks the array's
 * device address up (cudaGetSymbolAddress, with that device current), so make that one outside a stream capture.  All
 * calls on a device share the array: it keeps the last call's contents (the counters are cleared at the start of each
 * call, the bodies are rewritten up to n and not read beyond), and two calls that overlap on the GPU (different streams
 * without an ordering between them) race on it; so do calls from several host threads at once.
 * P3T_ECAPACITY: n > P3T_STATIC_MAX_N (nothing is launched).  P3T_EINVAL: n = 0, a null mass / pos / acc / pot, device
 * outside 0..63, eps < 0, not (0 <= r_in < r_out <= r_search), non-finite parameters.  P3T_ECUDA: a CUDA call failed.
 * The message of the last failure: p3t_direct_static_last_error() (process-wide, not thread-safe). */
#define P3T_STATIC_MAX_N 65536
p3t_status p3t_direct_static(int device, void *cuda_stream, size_t n, const float *mass, const float *pos, float eps,
                             float r_in, float r_out, float r_search, float *acc, float *pot, uint32_t *nbr_count,
                             uint64_t *info);
const char *p3t_direct_static_last_error(void);

/* acc[3n] (x,y,z interleaved) and pot[n], user order.  Either may be NULL. */
p3t_status p3t_get_acc_pot(p3t_ctx *ctx, float *acc, float *pot, int on_device);

/* count[n] list lengths in user order (may be NULL) and *total [host]
 * (may be NULL; reading it synchronises). */
p3t_status p3t_get_neighbour_counts(p3t_ctx *ctx, uint32_t *count, uint64_t *total, int on_device);

/* CSR: offset[n+1], nbr[capacity] in user ids, self excluded, each list sorted
 * ascending.  P3T_ECAPACITY if the lists do not fit `capacity` or the context's
 * nbr_capacity (offset is still written). */
p3t_status p3t_get_neighbours(p3t_ctx *ctx, uint64_t *offset, uint32_t *nbr, size_t capacity, int on_device);

/* Synchronises the stream, then reports counts and per-phase times (CUDA events). */
p3t_status p3t_get_stats(p3t_ctx *ctx, p3t_stats *out);

/* Hard part over the neighbour lists (the NEXT row of SURVEY.md 8(f); the paper evaluates it on the host,
 * PAPER.md L138, procedure step 3 L147).  For every particle i, from the lists L_i of the last p3t_eval_soft
 * (or p3t_eval_direct) and the positions and masses loaded then:
 *   acc[3n]   a_i   = - sum_{j in L_i} m_j (1 - K(s_ij)) q_ij / s_ij^3        (Eq. 7, per unit mass)
 *   jerk[3n]  d a_i / dt for relative velocities v_ij = vel_i - vel_j           (input of the Hermite scheme)
 *   pot[n]    phi_i = - sum_{j in L_i} m_j (1 - W(s_ij)) / s_ij                 (Eq. 5)
 * Since 1 - K = 1 - W = 0 beyond r_out <= r_search these equal the sums over all j.  vel[3n] is in user order,
 * interleaved like pos; outputs are double precision (every pair is evaluated in fp64), user order; any output
 * may be NULL.  vel and the outputs are all host or all device (on_device); the host form synchronises.
 * P3T_ESTATE before an eval call; P3T_ECAPACITY if the lists did not fit nbr_capacity (outputs untouched;
 * in the device form the error surfaces at the next synchronising call); P3T_EINVAL for null or non-finite vel. */
p3t_status p3t_eval_hard(p3t_ctx *ctx, const float *vel, double *acc, double *jerk, double *pot, int on_device);

/* Statistics of the Hermite part of one soft step. */
typedef struct {
    uint64_t n_nonisolated;  /* particles with a non-empty neighbour list (integrated by the Hermite scheme) */
    uint64_t n_blocks;       /* block steps of the neighbour cluster that needed most (clusters keep their own block times) */
    uint64_t n_steps;        /* Hermite steps summed over particles (N_step of Eq. 21) */
    uint64_t floor_hits;     /* times the criterion asked for less than one tick (dt_soft / 2^40) */
    uint64_t n_components;   /* neighbour clusters: connected components of the neighbour graph */
    uint64_t max_component;  /* particles in the largest one */
    float ms;                /* device time of the Hermite part incl. the drift of the isolated particles */
} p3t_hermite_info;

/* One soft step under H_hard (the NEXT row of SURVEY.md 8(f), rank 2; procedure step 3; steps 5-6 of the
 * GPU procedure in section 2.2, which the paper runs on the host).  pos[3n], vel[3n] (double, user order, interleaved)
 * are advanced in place over dt_soft: particles whose list of the last evaluation is empty ("isolated") drift,
 * pos += dt_soft vel; the others are integrated with the fourth-order Hermite scheme with block timesteps, their force
 * being Eq. 7 (L63) over their list with the masses loaded for that evaluation, every pair in fp64.
 *   - time runs in ticks of dt_soft / 2^40; a step is a power of two of ticks, at most dt_soft / 2^log2_div
 *     (Delta t_max, L158), the largest not above the criterion that divides the particle's current time;
 *   - first step: Eq. 20 (L163) with eta_s; afterwards Eq. 18 (L152) with eta, read as Aarseth's criterion with
 *     |a| -> sqrt(|a|^2 + a0^2) (A22); a2, a3 from the Hermite interpolation;
 *   - a0 = alpha m / r_cut^2 (Eq. 19) is the caller's to compute; with a0 = 0 the criterion collapses when a
 *     neighbour sits at the cutoff radius and the call ends with P3T_ELIMIT after max_blocks blocks (pos, vel are
 *     then mid-step and must be discarded).
 * The lists must be symmetric (j in L_i <=> i in L_j) and complete: that holds for p3t_eval_soft on an unsharded
 * context and for p3t_eval_direct over all particles; after a sharded evaluation (p3t_set_shard with world > 1) or a
 * subset p3t_eval_direct the call returns P3T_ESTATE, and the symmetry is checked on the device besides (P3T_ESTATE,
 * whatever the size of the cluster).  pos and vel are both host or both device (on_device); the call synchronises either
 * way (info is filled; may be NULL).
 * P3T_ESTATE before an eval call; P3T_ECAPACITY if the lists did not fit nbr_capacity; P3T_EINVAL for bad arguments
 * and when a force came out non-finite (coincident particles with eps = 0): pos, vel are then unusable. */
p3t_status p3t_hermite_step(p3t_ctx *ctx, double *pos, double *vel, double dt_soft, int log2_div, double eta, double eta_s,
                            double a0, long long max_blocks, int on_device, p3t_hermite_info *info);

/* Accuracy parameters of the Hermite part for particles of class 1 (black holes) when pair classes are set: eta and
 * eta_s as in p3t_hermite_step (a value <= 0: the call's own), a0 (< 0: the call's own).  L287: "The accuracy parameter
 * of timestep criterion for FS eta_FS is 0.1, and for SMBH eta_BH is 0.03"; a0 = alpha m / r_cut^2 (Eq. 19) differs with
 * the mass and the cutoff radius of the class.  P3T_EINVAL for non-finite values. */
p3t_status p3t_set_hermite_class_params(p3t_ctx *ctx, double eta_bh, double eta_s_bh, double a0_bh);

/* Tuning knob of p3t_hermite_step: the largest neighbour cluster (connected component of the lists) that one thread-block
 * cluster of 8 CTAs integrates with its own block times; still larger ones go together through a cooperative kernel
 * with grid barriers.  Components of up to 64 particles always take one warp each.  Default 4096; 64..1048576.
 * Results do not depend on it beyond rounding of nothing: the arithmetic per particle is the same. */
p3t_status p3t_set_hermite_cluster_max(p3t_ctx *ctx, int max_members);

/* One step of the scheme (L142-153) on a state the caller keeps in double precision: velocity kick by dt_soft / 2 with
 * the soft acceleration of the last evaluation (step 2), p3t_hermite_step (step 3), then positions rounded to float,
 * p3t_load_particles + p3t_build_tree + p3t_eval_soft at the new time and the second kick (step 4).  Before the first
 * step the caller loads the float-rounded positions and calls p3t_eval_soft once; afterwards the context always holds
 * the soft force and the lists of the current positions.  mass[n] float as in p3t_load_particles; mass, pos, vel are
 * all host or all device.  Errors as for the calls it is made of; P3T_ESTATE on a sharded context (the kick needs the
 * soft force of all particles, the Hermite part their lists). */
p3t_status p3t_step(p3t_ctx *ctx, const float *mass, double *pos, double *vel, double dt_soft, int log2_div, double eta,
                    double eta_s, double a0, long long max_blocks, int on_device, p3t_hermite_info *info);

/* Wait for all enqueued work; returns deferred device-side errors. */
p3t_status p3t_synchronize(p3t_ctx *ctx);

const char *p3t_last_error(const p3t_ctx *ctx);

/* Calibration of the ALU roofline denominator (not part of the hot path):
 * runs a pure-FFMA kernel (packed = 0: scalar FFMA, 1: packed FFMA2; 2, 3, 4: FFMA2 whose sources
 * are three distinct register pairs / pair x scalar-broadcast + pair / two distinct pairs -- the
 * register-operand bandwidth test of profiles/ffma2_operand_bandwidth_r1.md) of `iters` outer
 * iterations on the context's stream, synchronises, and returns the best of four timed
 * launches as TFLOP/s (2 flop per fp32 FMA) in *tflops [host] and its duration in *ms
 * [host, nullable].  P3T_EINVAL for null ctx/tflops, iters <= 0 or packed outside 0..7 (5, 6: the operand patterns of modes 2, 3 issued as scalar FFMAs; 7: mode 2 with one source shared by consecutive instructions). */
p3t_status p3t_measure_fp32_peak(p3t_ctx *ctx, int packed, int iters, double *tflops, float *ms);

/* Latency probes behind the floor table of the a1-a6 chain (profiles/tree_latency_floor_r2.md; not part of the hot path):
 * ns per step of `iters` dependent steps of  what = 0: loads that hit L2;  1: global atomics;  2: back-to-back launches
 * of an empty kernel;  3: the same launched with programmatic dependent launch;  4: fence + atomic + L2 load (one level
 * of the moments climb).  Uses the first 32 MiB of the workspace as scratch: the context must be loaded again afterwards
 * (P3T_ENOMEM if the workspace is smaller).  Synchronises.  P3T_EINVAL for bad arguments. */
p3t_status p3t_measure_latency(p3t_ctx *ctx, int what, int iters, double *ns);

/* Inspection of intermediate arrays (for the a1-a6 parity tests).  Valid after
 * p3t_build_tree.  p3t_array_info gives element count and element size. */
typedef enum {
    P3T_ARR_ROOT_CUBE   = 0,  /* float[4]: min corner x,y,z and side */
    P3T_ARR_KEYS        = 1,  /* uint64[n]: sorted Morton keys */
    P3T_ARR_SORTED_IDX  = 2,  /* uint32[n]: sorted position -> user id */
    P3T_ARR_BODIES      = 3,  /* float4[n]: sorted (x,y,z,m) */
    P3T_ARR_CELL_MAC    = 4,  /* float4[n_cells]: centre of mass, squared acceptance radius */
    P3T_ARR_CELL_MOM0   = 5,  /* float4[n_cells]: M, Qxx, Qyy, Qzz (traceful, about the COM) */
    P3T_ARR_CELL_MOM1   = 6,  /* float4[n_cells]: Qxy, Qxz, Qyz, bounding radius about the COM (with pair classes its
                                 sign bit marks the cells that hold a black hole) */
    P3T_ARR_CELL_META   = 7,  /* uint32[2][n_cells]: leaf: body start, count | 0x80000000;
                                                     internal: first child, child count */
    P3T_ARR_CELL_LEVEL  = 8,  /* uint8[n_cells] */
    P3T_ARR_CELL_START  = 9,  /* uint32[n_cells]: first body (sorted position) of the cell */
    P3T_ARR_CELL_PARENT = 10, /* uint32[n_cells] (root: 0xffffffff) */
    P3T_ARR_GROUP_START = 11, /* uint32[n_groups + 1] */
    P3T_ARR_CELL_BMIN   = 12, /* float4[n_cells]: tight AABB min of the cell's bodies */
    P3T_ARR_CELL_BMAX   = 13, /* float4[n_cells] */
    P3T_ARR_GROUP_STATS = 14, /* uint32[4][n_groups], valid after p3t_eval_soft: p-p list length,
                                 p-c list length, start and end of the group's walk in ns
                                 (low 32 bits of %globaltimer) -- load-balance diagnostics */
    P3T_ARR_GROUP_ORDER = 15  /* uint32[n_groups], valid after p3t_eval_soft: the groups by decreasing cost of that
                                 walk (13 x p-p + 33 x p-c list length, doubled for groups of more than 32 bodies; sorted by
                                 cost class, eight classes per octave, any order inside a class);
                                 the next p3t_eval_soft hands the groups to the warps in this order */
} p3t_array;
p3t_status p3t_array_info(p3t_ctx *ctx, p3t_array which, size_t *count, size_t *elem_bytes);
p3t_status p3t_copy_array(p3t_ctx *ctx, p3t_array which, void *dst, size_t dst_bytes, int on_device);

#ifdef __cplusplus
}
#endif
#endif /* P3T_H */
