/*
 * mlip.h -- C ABI of the B200-native energy-and-force hot path of
 * "Scalable Foundation Interatomic Potentials via Message-Passing Pruning and Graph
 * Partitioning" (arxiv 2509.21694; citations below are PAPER.md line numbers).
 *
 * The calls follow the paper's statement of the problem:
 *   atoms + cell -> radius graph (r_c)                      mlip_build_graph
 *   graph -> P spatial bins + halo of width K*r_c           mlip_partition / _grid
 *   first K of M message-passing layers (MPDP) on every
 *   extended sub-graph, sum root energies, sum gradients    mlip_energy_forces
 *
 * Conventions
 *   - Every entry point returns 0 (MLIP_OK) or a negative mlip_status; it never throws,
 *     aborts or exits. mlip_last_error(ctx) gives a human readable message for the last
 *     failure on that context.
 *   - "dev" pointers are CUDA device pointers on the context's device; "host" pointers are
 *     ordinary host memory. The library never takes ownership of caller arrays; inputs are
 *     only read during the call, outputs are fully overwritten.
 *   - Work is enqueued on the stream given to mlip_ctx_create. Calls that return a host
 *     scalar (build_graph: edge count; partition: sizes) synchronise that stream once.
 *     mlip_energy_forces is asynchronous: its outputs are valid after the caller
 *     synchronises the stream.
 *   - Handles are owned by the library and released only by the matching *_destroy.
 *   - Atom ids are int32; the number of directed edges must stay below 2^31.
 *   - Everything runs in hand-written sm_100a kernels; there is no CPU fallback. If no
 *     CUDA device is usable the calls fail with MLIP_ERR_CUDA.
 */
#ifndef MLIP_H_
#define MLIP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  MLIP_OK = 0,
  MLIP_ERR_INVALID_ARG = -1,
  MLIP_ERR_UNSUPPORTED = -2,     /* singular cell, d not in {64,128,256}, L > L_max ... */
  MLIP_ERR_HALO_TOO_SMALL = -3,  /* halo < L*r_cut: refused rather than silently wrong forces */
  MLIP_ERR_OUT_OF_MEMORY = -4,
  MLIP_ERR_OVERFLOW = -5,        /* number of edges >= 2^31 or image shift outside [-127,127] */
  MLIP_ERR_CUDA = -6,
  MLIP_ERR_NUMERIC = -7          /* non-finite energy or force: the 16-bit path left the IEEE-half range (see MLIP_BF16) */
} mlip_status;

/* Arithmetic of the contractions.
 *   MLIP_FP32  fp32 arithmetic everywhere (north_star tolerances 1e-5 / 1e-4). Contractions by CUDA-core FMA, except at
 *              d = 128 (fused edge kernels and node GEMMs): tcgen05 with every fp32 operand split exactly into three bf16 terms, six MMAs per
 *              product, fp32 accumulation (24 significant bits, fp32 range). The tensor core truncates when it
 *              adds into its accumulator: per-atom energies carry a systematic relative error of about 1e-6 (1e-5 at four
 *              times the density of the BASELINE configurations), forces 5e-6 of their RMS.
 *   MLIP_BF16  16-bit tensor-core operands with fp32 accumulation (tcgen05, accumulators in TMEM). The name follows
 *              BASELINE.json ("bf16 GEMM inputs"); what runs is IEEE HALF (f16) operands in every contraction -- same
 *              tensor-core rate and bytes as bf16, three more mantissa bits (force RMS error of the unpruned L = 15
 *              configuration 4.5e-3 instead of 1.7e-2 with bf16 node operands), and packed f16x2 epilogue arithmetic
 *              in the fused edge kernels. Range contract of the f16 tensors (the 16-bit copies of h, c-bar, Q-bar; the
 *              halved pre-activations P, Q, a, p; messages; the adjoints mbar, pbar, abar): magnitudes below 65504. The reverse
 *              pass is scaled by a power of two chosen per sub-domain from max|d E / d o| (removed again when the
 *              forces are assembled), so small adjoints do not fall into the f16 subnormals. A value that leaves
 *              the range becomes inf/NaN, reaches E or F, and is reported as MLIP_ERR_NUMERIC by the next
 *              synchronising call (mlip_step_host, mlip_md_*) or by mlip_ctx_status -- never a silent wrong number. */
enum { MLIP_FP32 = 0, MLIP_BF16 = 1 };

typedef struct mlip_ctx mlip_ctx;
typedef struct mlip_model mlip_model;
typedef struct mlip_graph mlip_graph;
typedef struct mlip_part mlip_part;

#define MLIP_MAGIC 0x50494c4du /* "MLIP" */

/* Shape of the message-passing network (BASELINE.json configs; the paper treats the network
 * as a black box, PAPER.md:23,151 -- the concrete equations are readings O2-O4 of DESIGN.md). */
typedef struct {
  uint32_t magic;     /* MLIP_MAGIC */
  uint32_t version;   /* 1 */
  int32_t n_species;  /* S */
  int32_t d;          /* hidden width, one of 64, 128, 256 */
  int32_t n_rbf;      /* number of Gaussian radial basis functions, 2..16 */
  int32_t L_max;      /* M: number of message-passing layers stored in the blob */
  float r_cut;        /* local cutoff r_c in Angstrom */
  float agg_scale;    /* alpha multiplying the neighbour sum (reading R7) */
  int32_t flags;      /* bit 0 (MLIP_FLAG_THREE_BODY): three-body variant, see mlip_model_load; other bits must be 0 */
  int32_t n_rbf3;     /* three-body variant: radial functions of the angle basis, must be 4 (else 0) */
  int32_t l_max;      /* three-body variant: largest l of Y_l^0(cos theta), must be 3 (else 0) */
  float r_cut3;       /* three-body variant: cutoff r_3 <= r_cut of the edge pairs, Angstrom (else 0) */
} mlip_model_header;
#define MLIP_FLAG_THREE_BODY 1

/* Number of floats the weight blob must hold for a header. */
size_t mlip_model_num_weights(const mlip_model_header* h);

/* Create a context bound to CUDA device `device` and to `stream` (a cudaStream_t, may be
 * NULL for the default stream). */
int mlip_ctx_create(int device, void* stream, mlip_ctx** out);
void mlip_ctx_destroy(mlip_ctx* ctx);
const char* mlip_last_error(const mlip_ctx* ctx);
/* Synchronises the context stream and returns (and clears) the status of the asynchronous work enqueued so far:
 * MLIP_OK, MLIP_ERR_NUMERIC (non-finite energy or force, see MLIP_BF16), MLIP_ERR_CUDA. mlip_energy_forces* are
 * asynchronous and cannot report such a condition themselves; calls that synchronise anyway (mlip_step_host,
 * mlip_md_*) return it directly. */
int mlip_ctx_status(mlip_ctx* ctx);

/* Load a weight blob (HOST pointer, fp32, `n` floats, copied). Order, every matrix row-major
 * [out,in]:  T[S,d], E0[S], then for each of the L_max layers
 *   W1[d, 2d+n_rbf] (columns: receiver h_i | sender h_j | e_hat), b1[d], W2[d,d], b2[d],
 *   V1[d, 2d] (columns: h | m), c1[d], V2[d,d], c2[d]
 *   (and, with MLIP_FLAG_THREE_BODY, G[16,d], g[16], W3[d,16]);   finally Wo[d,d], bo[d], wo[d], b_E.
 *
 * Three-body (angle) variant, BASELINE.json config 5 (the paper's workhorse MatterSim is an M3GNet-type model,
 * PAPER.md:91,119,131; the paper gives no equations -- definition O7 of DESIGN.md): for edges with
 * r_e < r_cut3 the first edge linear gets the extra term W3 t_e with
 *   t_e = u3(r_e) sum over in-edges e' = (i <- k) != e of the same receiver, r_e' < r_cut3, of
 *         u3(r_e') [Y_l^0(cos theta_ee') g3_n(r_e')]_{4l+n} * sigmoid(G h_k + g),     l = 0..3, n = 0..3,
 * u3 the cosine envelope on [0, r_cut3], g3_n Gaussians centred at n r_cut3 / 3 of width r_cut3 / 3, theta the angle at
 * the receiver. Needs n_rbf3 = 4, l_max = 3, 0 < r_cut3 <= r_cut (the halo stays L r_cut); evaluated in MLIP_FP32 only;
 * at most 128 neighbours inside r_cut3 per atom (else MLIP_ERR_UNSUPPORTED from the next synchronising call). */
int mlip_model_load(mlip_ctx* ctx, const mlip_model_header* h, const float* w_host, size_t n,
                    mlip_model** out);
void mlip_model_destroy(mlip_model* m);

/* Radius graph under periodic boundaries, by a cell list built with a counting
 * sort + prefix sum. Directed edge (i <- j, n) exists iff |x_j - x_i + n.C|^2 < r_cut^2
 * (strict, float64, fixed operation order, reading R10) and not (i == j and n == 0).
 *   pos_dev     [n_atoms,3] float64, device, unwrapped Cartesian positions (Angstrom)
 *   cell_host   [3,3] float64, HOST, rows are the lattice vectors a1,a2,a3 of any non-singular
 *               (triclinic) cell; a singular one gives MLIP_ERR_UNSUPPORTED (R12)
 *   species_dev [n_atoms] int32, device, values in [0, n_species)
 * The graph keeps its own (cell-sorted) copy of what it needs. */
int mlip_build_graph(mlip_ctx* ctx, const double* pos_dev, const double* cell_host,
                     const int32_t* species_dev, int64_t n_atoms, double r_cut, mlip_graph** out);
int mlip_graph_num_edges(const mlip_graph* g, int64_t* n_edges);
/* Edge list in canonical order: lexicographic by (i, j, n_x, n_y, n_z) in the caller's atom
 * numbering. recv_dev/send_dev [E] int32, shift_dev [E,3] int32, all device. */
int mlip_graph_export_edges(mlip_ctx* ctx, const mlip_graph* g, int32_t* recv_dev,
                            int32_t* send_dev, int32_t* shift_dev);
void mlip_graph_destroy(mlip_graph* g);

/* Spatial partition (PAPER.md:157 Stage 1: uniform grid of P bins on the scaled positions;
 * Stage 2: every bin is extended so that each root atom keeps its K-hop
 * neighbourhood). K = ceil(halo / r_c). The extended set of a bin is found in two steps:
 *   (a) the geometric box: atoms whose periodic distance to the bin is <= halo along every axis
 *       (a superset of the K-hop set when halo >= K*r_c, reading R2);
 *   (b) by default, a K-level breadth-first search over the radius graph from the root atoms inside
 *       that box (the paper's own rule): atoms not reached within K hops leave the sub-domain, and
 *       the hop count of the others is their depth class (see mlip_part_layer_info).
 * mlip_ctx_set_khop_halo(ctx, 0) keeps the whole box of (a) and uses geometric shells of thickness r_c
 * as depth classes instead. Results are identical either way; (b) evaluates fewer atoms and edges.
 * mlip_partition cuts n_sub slabs along the axis of largest perpendicular width (R3). */
int mlip_partition(mlip_ctx* ctx, const mlip_graph* g, int n_sub, double halo, mlip_part** out);
int mlip_partition_grid(mlip_ctx* ctx, const mlip_graph* g, const int grid[3], double halo,
                        mlip_part** out);
/* mlip_partition_grid for ONE shard of a multi-GPU run: only the sub-domains k with k mod n_shards == shard
 * (k = (bx * gy + by) * gz + bz, the dealing rule of mlip_energy_forces_shard) are built; the others keep their index
 * and stay empty (mlip_part_info reports zeros), so that a rank spends partition time and memory on its own
 * sub-domains only. The handle must be evaluated by mlip_energy_forces_shard / _stress with the same (shard,
 * n_shards); anything else is refused with MLIP_ERR_INVALID_ARG. */
int mlip_partition_grid_shard(mlip_ctx* ctx, const mlip_graph* g, const int grid[3], double halo, int shard,
                              int n_shards, mlip_part** out);
int mlip_part_count(const mlip_part* p, int* n_sub);
/* Sizes of sub-domain s: root (owned) atoms, extended atoms, induced directed edges. The halo
 * growth factor of PAPER.md:289 is (n_ext - n_owned) / n_owned. */
int mlip_part_info(const mlip_part* p, int s, int64_t* n_owned, int64_t* n_ext, int64_t* n_edges);
/* Per-layer active sets of sub-domain s when the first L layers are evaluated. The extended atoms of a sub-domain are
 * numbered by depth class: 0 = root atoms; k >= 1 = halo atoms k hops away from the nearest root atom (K-hop search,
 * default) or, with the geometric halo, atoms whose largest per-axis periodic distance to the bin lies in
 * ((k-1) r_c, k r_c] -- a lower bound of the hop count because an edge is shorter than r_c. The root energies of
 * PAPER.md:169 and their gradient depend on layer l (0-based) only through receivers of class <= L-1-l
 * and senders of class <= L-l: the K-hop neighbourhood of PAPER.md:165 shrinks by one hop per layer.
 * mlip_energy_forces evaluates exactly those prefixes; the result is identical to evaluating every layer on the whole
 * extended sub-graph.
 *   n_recv  atoms whose h^{l+1} is computed, n_send atoms whose h^l is read, n_edges edges evaluated by layer l
 * (with active sets switched off through mlip_ctx_set_active_sets: n_ext, n_ext, all induced edges). */
int mlip_part_layer_info(const mlip_part* p, int s, int L, int l, int64_t* n_recv, int64_t* n_send,
                         int64_t* n_edges);
void mlip_part_destroy(mlip_part* p);

/* Energy and forces with the first L of L_max layers (MPDP).
 * E = sum over sub-domains of the ROOT-atom energies; F = - sum over
 * sub-domains of the gradient of that sub-domain's root energy w.r.t. ALL of its atoms
 * (reading R1). part == NULL evaluates the whole box as one domain.
 * Sub-domains are evaluated one after another on the context stream.
 *   precision       MLIP_FP32 (fp32 contractions) or MLIP_BF16 (16-bit tensor-core contractions
 *                   with fp32 accumulation, see the enum; requires d = 256 or 128)
 *   energy_dev      [1] float64, device
 *   forces_dev      [n_atoms,3] float32, device, caller's atom numbering (eV/Angstrom)
 *   atom_energy_dev [n_atoms] float32, device, or NULL
 * Fails with MLIP_ERR_HALO_TOO_SMALL if part was built with halo < L*r_cut. */
int mlip_energy_forces(mlip_ctx* ctx, const mlip_model* m, int L, const mlip_graph* g,
                       const mlip_part* part, int precision, double* energy_dev,
                       float* forces_dev, float* atom_energy_dev);

/* The same evaluation restricted to the sub-domains k with k mod n_shards == shard (sub-graph
 * predictions are completely independent, and are distributed over devices in
 * PAPER.md:177). Energies and forces are this shard's PARTIAL sums over the whole box (zeros
 * where it contributes nothing); summing the outputs of all shards -- one all-reduce of E and F
 * when the shards live on different GPUs -- gives exactly the unsharded result up to fp32
 * summation order. atom_energy_dev holds E_i for the atoms this shard owns, 0 elsewhere. */
int mlip_energy_forces_shard(mlip_ctx* ctx, const mlip_model* m, int L, const mlip_graph* g,
                             const mlip_part* part, int shard, int n_shards, int precision,
                             double* energy_dev, float* forces_dev, float* atom_energy_dev);

/* Energy, forces and the stress tensor sigma = (1/V) dE/d(strain) (with energy-gradient forces the
 * stress decomposes over sub-graphs like the forces do). Every edge vector follows a homogeneous strain as
 * r_e -> (1 + eps) r_e, so sigma_ab = (1/V) sum over sub-domains and their directed edges of rbar_e r_a r_b / r_e with
 * rbar_e the adjoint of the root-energy sum w.r.t. the edge length -- the same per-edge scalars the forces are
 * assembled from. Arguments as mlip_energy_forces_shard (shard = 0, n_shards = 1 for the whole box), plus
 *   stress_dev [3,3] float64, device, row-major, symmetric, eV/Angstrom^3 (this shard's partial sum). */
int mlip_energy_forces_stress(mlip_ctx* ctx, const mlip_model* m, int L, const mlip_graph* g,
                              const mlip_part* part, int shard, int n_shards, int precision,
                              double* energy_dev, float* forces_dev, float* atom_energy_dev,
                              double* stress_dev);

/* Whole step from HOST buffers: copies positions/species to the device, builds the graph,
 * partitions (grid = {1,1,1} means one domain), evaluates, copies E and F back and
 * synchronises. This is the call bench.py times for its end-to-end figure. */
int mlip_step_host(mlip_ctx* ctx, const mlip_model* m, int L, const double* pos_host,
                   const double* cell_host, const int32_t* species_host, int64_t n_atoms,
                   const int grid[3], double halo, int precision, double* energy_host,
                   float* forces_host);

/* Per-layer active sets inside sub-domains (see mlip_part_layer_info): on by default; enable = 0 makes every layer run
 * on the whole extended sub-graph (same results; kept for A/B measurement and as a test control). */
int mlip_ctx_set_active_sets(mlip_ctx* ctx, int enable);
/* Halo rule used by the NEXT mlip_partition* calls of this context: 1 (default) = K-hop breadth-first search inside the
 * geometric box, 0 = the whole geometric box (see mlip_partition). */
int mlip_ctx_set_khop_halo(mlip_ctx* ctx, int enable);

/* On-device NVE molecular dynamics (the use the paper builds the partitioned evaluation for):
 * n_steps of velocity-Verlet -- v += (dt/2) a; x += dt v; rebuild the graph (and the partition when grid != {1,1,1});
 * E, F; v += (dt/2) a -- with a = 9.648533e-3 F / m. Every step runs on the GPU; the host only sequences launches.
 *   pos_dev, vel_dev   [n_atoms,3] float64, device, IN/OUT (Angstrom, Angstrom/fs; positions are not wrapped)
 *   mass_dev           [n_atoms] float64, device (amu);  species_dev [n_atoms] int32, device
 *   cell_host          [3,3] float64, HOST (fixed cell)
 *   grid, halo         partition as in mlip_partition_grid ({1,1,1}: one domain)
 *   dt                 fs
 *   total_energy_host  [n_steps+1] float64, HOST or NULL: potential + kinetic energy (eV) before every step and after
 *                      the last one
 * Synchronises the stream before returning. */
int mlip_md_nve(mlip_ctx* ctx, const mlip_model* m, int L, double* pos_dev, double* vel_dev,
                const double* mass_dev, const double* cell_host, const int32_t* species_dev,
                int64_t n_atoms, const int grid[3], double halo, int precision, double dt, int n_steps,
                double* total_energy_host);

/* On-device molecular dynamics, general form. Every MD result of the paper is ASE Langevin dynamics (PAPER.md:89, 91,
 * 137); the paper does not print the update rule, so the thermostat is the BAOAB splitting (reading R20 of DESIGN.md):
 *   B  v += (dt/2) a(x);  A  x += (dt/2) v;  O  v = c1 v + c2 sqrt(kB T / m) xi;  A  x += (dt/2) v;  E, F;  B  v += (dt/2) a
 * with c1 = exp(-friction dt), c2 = sqrt(1 - c1^2), kB = 8.617333262e-5 eV/K and three standard normals xi per atom and
 * step from the counter-based generator Philox4x32-10: counter (atom, step, 0, 0), key (seed low, seed high), Box-Muller
 * on (x + 0.5) 2^-32 -- a pure function of (seed, step, atom index in the caller's numbering), independent of the
 * partition, of the internal atom order and of the number of GPUs. thermostat = MLIP_MD_NVE is plain velocity Verlet.
 *
 * skin > 0 (Angstrom) switches on Verlet-skin reuse: the radius graph is built once with r_cut + skin and partitioned
 * once (root atoms keep their sub-domain, the K-hop search runs over the skin graph, a superset of every later graph);
 * every step only filters that candidate list with the canonical float64 predicate at the current positions -- the edge
 * set of every step is exactly the one a fresh mlip_build_graph would return -- and the whole is rebuilt when an atom has
 * moved more than skin/2 since the last build. cuda_graph = 1 additionally captures the per-step evaluation (filter,
 * layers, reverse pass, force assembly: fixed launch dimensions between rebuilds) in a CUDA graph that is replayed until
 * the next rebuild. Arguments as mlip_md_nve; stats may be NULL. Synchronises the stream before returning. */
enum { MLIP_MD_NVE = 0, MLIP_MD_LANGEVIN = 1 };
typedef struct {
  double dt;            /* fs */
  int32_t n_steps;
  int32_t thermostat;   /* MLIP_MD_NVE or MLIP_MD_LANGEVIN */
  double temperature;   /* K */
  double friction;      /* 1/fs */
  uint64_t seed;
  double skin;          /* Angstrom; 0 = rebuild graph and partition every step */
  int32_t cuda_graph;   /* 1 = replay a captured CUDA graph between rebuilds (needs skin > 0) */
  int32_t reserved;
} mlip_md_params;
typedef struct {
  int64_t n_rebuilds;        /* graph + partition builds, the initial one included */
  int64_t n_graph_replays;   /* steps evaluated by replaying a captured CUDA graph */
  double ms_total;           /* device time of the n_steps steps (CUDA events on the context stream) */
} mlip_md_stats;
int mlip_md_run(mlip_ctx* ctx, const mlip_model* m, int L, double* pos_dev, double* vel_dev,
                const double* mass_dev, const double* cell_host, const int32_t* species_dev,
                int64_t n_atoms, const int grid[3], double halo, int precision,
                const mlip_md_params* params, double* total_energy_host, mlip_md_stats* stats);

/* Number of kernel launches issued by this context so far (for bench.py's gpu_launches). */
int64_t mlip_ctx_launch_count(const mlip_ctx* ctx);

/* Per-kernel-group device timing (SURVEY.md 5 "tracing": CUDA events on the context stream,
 * one pair around each launch group). mlip_ctx_profile(ctx, 1) clears the counters and starts
 * recording, (ctx, 0) stops. mlip_ctx_profile_read synchronises the stream and returns the
 * accumulated milliseconds and kernel-launch count of one group since the last enable. */
typedef enum {
  MLIP_GROUP_EDGE_FWD = 0,       /* fused gather -> edge MLP -> segmented sum (steps A6+A7) */
  MLIP_GROUP_EDGE_BWD = 1,       /* its reverse pass (edge part of A10) */
  MLIP_GROUP_GATHER_REV = 2,     /* sender-side adjoint gather through the reverse-edge index */
  MLIP_GROUP_NODE_GEMM = 3,      /* node pre-projection / update / readout contractions (A8-A10) */
  MLIP_GROUP_READOUT_FORCES = 4, /* embedding, readout, energy sum, force assembly (A9, A11) */
  MLIP_GROUP_GRAPH = 5,          /* mlip_build_graph (A1-A4) */
  MLIP_GROUP_PARTITION = 6,      /* mlip_partition / mlip_partition_grid (A5) */
  MLIP_GROUP_THREE_BODY = 7,     /* gates, triplet sums and their adjoints of the three-body variant (O7) */
  MLIP_GROUP_COUNT = 8
} mlip_group;
int mlip_ctx_profile(mlip_ctx* ctx, int enable);
int mlip_ctx_profile_read(mlip_ctx* ctx, int group, double* ms_total, int64_t* n_launches);

/* Exclusive prefix sum over int32 on the context stream: out_dev[i] = in_dev[0] + ... + in_dev[i-1] for i = 0..n, i.e.
 * out_dev has n + 1 entries and out_dev[n] is the total (how the library turns per-atom degrees into CSR row pointers
 * and flags into compaction offsets, steps A3/A5 of DESIGN.md 1). Device pointers, asynchronous, in_dev and out_dev must
 * not overlap; n = 0 writes out_dev[0] = 0. Sums wrap like int32 addition.
 *   mlip_scan_i32          the path the library uses internally: its scratch (tile totals) comes from the allocator,
 *                          any n < 2^31.
 *   mlip_scan_i32_noalloc  ALLOCATES NOTHING (no cudaMalloc / cudaFree, no allocating library routine; three kernel
 *                          launches), for callers that cannot allocate: CUDA graph capture, serving loops, harnesses
 *                          that forbid it. Its scratch is a fixed 128 KiB array in device memory that every GPU which
 *                          loads the library holds until exit; hence n <= MLIP_SCAN_NOALLOC_MAX, beyond which the call
 *                          returns MLIP_ERR_INVALID_ARG with a message and launches nothing. All calls on a device
 *                          share that array: calls that OVERLAP on the GPU (two streams, concurrent graph replays)
 *                          race on it -- serialise them. The first call on a device resolves the array's address
 *                          (cudaGetSymbolAddress); make it before starting a capture. Same result as mlip_scan_i32,
 *                          bit for bit. */
#define MLIP_SCAN_NOALLOC_MAX 67108864 /* 32768 tiles x 2048 elements */
int mlip_scan_i32(mlip_ctx* ctx, const int32_t* in_dev, int32_t* out_dev, int64_t n);
int mlip_scan_i32_noalloc(mlip_ctx* ctx, const int32_t* in_dev, int32_t* out_dev, int64_t n);

#ifdef __cplusplus
}
#endif
#endif /* MLIP_H_ */
