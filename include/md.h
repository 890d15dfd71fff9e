/*
 * md.h -- C ABI of libmd_b200: the neighbor-list molecular-dynamics hot path of
 * "JAX, M.D." (arXiv 1912.04232) as hand-written CUDA kernels for sm_100a.
 *
 * Citations are lines of /root/reference/PAPER.md (L<line>, section); readings
 * of points the paper leaves open are SURVEY.md §8c A1..A18, restated in
 * DESIGN.md §3.
 *
 * Conventions (all calls)
 *   - Return value: MD_OK, or a negative MD_E* for a failure detected on the
 *     host before anything is launched; md_last_error() gives the text.
 *     Asynchronous conditions (list overflow, rebuild needed) are DEVICE words,
 *     never return codes.  No exceptions, no abort, no output to stdout.
 *   - Pointers are DEVICE pointers unless the parameter says "host".  The
 *     caller owns every buffer, the workspace included; the library allocates
 *     no caller-visible memory and keeps no pointer past a call except the
 *     workspace and (md_nve_step and the other step calls) a cached CUDA graph of
 *     the last call's arguments.  No call except md_create / md_destroy /
 *     md_nve_run_host synchronises with the host.  No behaviour depends on
 *     environment variables: every knob is an md_set_option.
 *   - A call makes the device that owns the workspace current on the calling thread for
 *     its own duration and restores the caller's current device before it returns.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default
 *     stream).  Work is ordered on that stream only.
 *   - Particle arrays are float4[n], 16-byte aligned:
 *       pos   = (x, y, z, w)  0 <= x < box[k]; z ignored (keep 0) when dim = 2;
 *               w = particle diameter d_i (MD_KIND_SOFT) or unused (MD_KIND_LJ)
 *       vel   = (vx, vy, vz, unused)
 *       force = (Fx, Fy, Fz, e_i)  with e_i = 1/2 sum_j u(r_ij) on output
 *     Indices are int32.
 */
#ifndef MD_B200_H
#define MD_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MD_OK          0
#define MD_EINVAL     (-1)  /* null/unaligned pointer, n<=0, dim not 2|3, capacity<=0 or not a
                               multiple of 4, skin<0, r_cut<=0, dt<=0, mass<=0, epsilon<=0, unknown kind or option */
#define MD_EBOX       (-2)  /* a box side holds fewer than 3 cells of side >= r_cut+skin, or the
                               cell side exceeds r_cut+skin by less than 1e-5 of the box side */
#define MD_EWORKSPACE (-3)  /* workspace null, unaligned (256 B) or too small */
#define MD_ECUDA      (-4)  /* CUDA runtime error at launch; text in md_last_error() */

#define MD_KIND_LJ   0      /* Lennard-Jones [69], L104 §3.3.2 */
#define MD_KIND_SOFT 1      /* harmonic soft sphere [70], L104; d_ij = (d_i+d_j)/2, L301 App. A */
#define MD_KIND_MORSE 2     /* Morse [75], L104: u = eps (1 - exp(-alpha (r - sigma)))^2 - eps */
#define MD_KIND_LJ_SPECIES 4 /* LJ with eps, sigma, r_cut per species pair (md_set_species_lj); species = (int)pos.w */
#define MD_KIND_BKS 5        /* exp-6 per species pair + damped shifted-force Coulomb (md_set_species_bks) */
#define MD_KIND_BUCKINGHAM 3 /* Buckingham-type exp-6 [71-73], L104: u = eps exp(-alpha r) - sigma / r^6
                               (epsilon = A, alpha = B, sigma = C) */

typedef struct md_system md_system;   /* opaque; lives in host memory */

/* Space + partitioning parameters (L72 §3.2.1 space.periodic(L); L84 §3.2.3). */
typedef struct md_config {
    int   dim;        /* 2 or 3 */
    float box[3];     /* periodic box sides L_k; box[2] ignored when dim = 2 */
    float r_cut;      /* neighborhood size sigma of L84 before the halo */
    float skin;       /* halo (L49 §3.1); list radius R = fl32(r_cut + skin) */
    int   capacity;   /* slots per neighbor row (static shape, L47 §3.1); multiple of 4 */
    int   resort;     /* 1: md_cell_list_build physically re-orders pos/vel/id by cell */
} md_config;

/* Pair potential u(r) (L78 §3.2.2, L104 §3.3.2). */
typedef struct md_potential {
    int   kind;       /* MD_KIND_LJ | MD_KIND_SOFT | MD_KIND_MORSE | MD_KIND_BUCKINGHAM | MD_KIND_LJ_SPECIES |
                         MD_KIND_BKS (the last two read their tables from md_set_species_lj / _bks) */
    float epsilon;
    float sigma;      /* LJ length; unused for SOFT (diameters come from pos.w) */
    float r_cut;      /* truncation radius (<= config r_cut); unused for SOFT, whose cutoff is the pair's own
                         d_ij = (d_i + d_j) / 2: the caller keeps every d_ij <= config r_cut (the list radius),
                         a larger overlap range is cut at the list (not checked: diameters are device data) */
    int   shift;      /* LJ, MORSE: 1 = u(r) - u(r_cut) for r < r_cut, 0 = plain truncation */
    float alpha;      /* MORSE: inverse width; sigma is its r0, epsilon its well depth D. Unused otherwise */
} md_potential;

/* Text of the last error on the calling thread ("" if none). Host pointer, valid until the
 * next failing call. */
const char *md_last_error(void);

/* Bytes of device workspace md_create needs for n particles (host out-pointer). */
int md_workspace_bytes(const md_config *cfg, int n, size_t *bytes);

/* Bind a system to a caller-owned device workspace (256-byte aligned, >= md_workspace_bytes).
 * Validates cfg (MD_EINVAL / MD_EBOX), clears the workspace on the legacy stream and
 * synchronises once.  *out is a host object released by md_destroy. */
int md_create(const md_config *cfg, int n, void *workspace, size_t bytes, md_system **out);
int md_destroy(md_system *sys);

/* Tuning knobs (host call; drops the cached step graph):
 *   "fast32"               1 (default): 3-D LJ, Morse and Buckingham forces by the fp32 fast path with
 *                          an error estimate and fp64 re-evaluation of the particles that need it
 *                          (DESIGN.md §5); 0: every pair in fp64 (the kernels selected by
 *                          threads_per_particle), as SOFT, LJ_SPECIES, BKS and every 2-D system always
 *   "est_thr"              the fast path re-evaluates particle i in fp64 when S_i, the root of the sum
 *                          over j of the squared error scale of pair ij (LJ: |f_ij|, floored near its
 *                          zero; Morse and Buckingham: the parts of f_ij times the amplification of
 *                          their exponentials, scaled to LJ's), exceeds est_thr * max(|F_i|, 1e-3);
 *                          default 3.5
 *   "threads_per_particle" fp64 force kernel variant: 0 = streaming kernel (one lane per particle,
 *                          list rows staged through shared memory by TMA; default for
 *                          n >= 32768), or 1, 2, 4 lanes sharing one particle (default 4 below)
 *   "fused"                1 (default): inside md_nve_step's graph the 3-D LJ force kernel also opens
 *                          the next step (second half-kick, first half-kick, drift into a second
 *                          position buffer, half-skin test); 0: k_kick_drift every step.  Same bits.
 *   "remap"                3-D LJ force kernel: blocks i and i + remap work on adjacent list tiles, so the
 *                          blocks one SM receives round-robin share gathered positions in L1 (default
 *                          a quarter of the device's SM count; 0 = block i works on tile block i)
 *   "builder_parts"        warps that share one list tile in the builder: 1, 2, 4, or 0 (default) = 4 up to
 *                          65,536 particles, else 1
 *   "builder"              neighbor-list kernel: 2 (default) records hits in per-lane bit masks,
 *                          1 appends them to per-lane shared-memory columns (first design)
 *   "cell_coop"            1: the cell list as ONE cooperative launch (grid barriers between its phases), 0: five
 *                          kernels; default 1 up to 65,536 particles (where it is faster), else 0.  Same results.
 *                          (The step loops use the cooperative form on their own account, "rebuild_flagged".)
 *   "use_graph"            0: the step calls launch their kernels directly instead of CUDA graphs -- the same
 *                          kernels in the same order (so a profiler lists them one by one); the rebuild kernels
 *                          are then launched every step and return at once while the step's device flag is 0
 *   "rebuild_flagged"      how the step loops (md_nve_step and the other rules) run the rebuild inside their CUDA
 *                          graphs.  1: two launches, the cooperative cell list and the neighbor-list builder, that
 *                          are part of every step and return at once while the step's device flag is 0 (2.7 us
 *                          each on B200); 0: the rebuild's kernels inside an IF node, which costs 9 us per step
 *                          whether or not it fires; -1 (default): 1 up to 600,000 particles (beyond that the
 *                          cooperative cell list loses more per rebuild than the IF node costs).  Same results.
 *   "step_fork"            1 (default): in md_nve_step's fused loop (3-D LJ, Morse, Buckingham with "rebuild_flagged"
 *                          in effect) the flagged rebuild runs on a branch BESIDE the force kernel instead of in
 *                          front of it: the branch holds the rebuild and a second launch of the force kernel that
 *                          runs only if the step's flag is up, the main branch the force kernel that runs only
 *                          if it is not; a step without a rebuild no longer waits for launches that do nothing
 *                          (74.6 -> 73.2 us per step at 256,000 particles).  0: in series.  Same results.
 *   "nh_chain"             thermostats in md_nose_hoover_step's chain, 1 (default) .. 8 */
int md_set_option(md_system *sys, const char *name, double value);

/* The value in effect: "rebuild_flagged" (1 or 0: what the step loops will do), "est_thr", "fast32",
 * "use_graph", "step_fork", "threads_per_particle".  Errors: MD_EINVAL (NULL, unknown name). */
int md_get_option(md_system *sys, const char *name, double *value);

/* Species x species Lennard-Jones tables (L104 pair potentials with per-species parameters; the
 * sigma matrix of L298-L305): host float[nspecies * nspecies], row-major, 1 <= nspecies <= 4, every
 * r_cut <= the list r_cut.  Used by MD_KIND_LJ_SPECIES (whose epsilon / sigma / r_cut fields are
 * ignored; shift applies per pair); the species of a particle is (int)pos.w.  fp64 pair chain. */
int md_set_species_lj(md_system *sys, int nspecies, const float *epsilon, const float *sigma,
                      const float *r_cut);

/*
 * Multi-GPU by replicated positions and a split neighbor list: every rank holds
 * all positions and runs the same cell list and re-sort, but builds list rows and computes forces only for
 * its own range of (cell-sorted) particles, integrates those, and the ranks exchange their position ranges
 * every step (velocities at rebuilds).  The list -- 4 * capacity bytes per particle against 16 for a
 * position -- is what is split.
 *
 * md_set_range (needs a system created with resort = 1: a range is a range of the cell-sorted order; MD_EINVAL
 * otherwise): this context owns particles [begin, end): begin a multiple of 32 (a list tile), end a
 * multiple of 32 or n.  From then on md_neighbor_list_build writes rows, counts and rebuild references of
 * that range only, md_pair_energy_force forces, e_i and the energy sum of that range only; md_cell_list_build stays global; the step calls (md_nve_step, ...) return MD_EINVAL -- the
 * step is driven from outside with the two calls below around the exchange.  [0, n) restores the default.
 */
int md_set_range(md_system *sys, int begin, int end);

/* First half of a velocity-Verlet step on the context's range: v += dt/(2m) F; r = wrap(r + dt v); *flag
 * (DEVICE int32) = 1 if a particle of the range is now more than skin/2 from its position at the last list
 * build, else 0.  The arithmetic of md_nve_step's own opening kernel. */
int md_kick_drift(md_system *sys, void *pos, void *vel, const void *force, float dt, float mass,
                  int32_t *flag, void *stream);

/* Second half of a velocity-Verlet step on the context's range in one launch: F = F(pos) over the list (no
 * energies: force.w = 0), then v += dt/(2m) F in the force kernel's epilogue -- md_nve_step's own closing
 * kernel.  Arguments as md_pair_energy_force, plus vel float4[n] in/out. */
int md_force_half_kick(md_system *sys, const md_potential *pot, const void *pos, const int32_t *nbr_idx,
                       const int32_t *nbr_count, void *force, void *vel, float dt, float mass, void *stream);

/* Closing half-kick on the context's range: v += dt/(2m) F. */
int md_half_kick(md_system *sys, void *vel, const void *force, float dt, float mass, void *stream);

/*
 * Multi-GPU by spatial decomposition: slabs along x with halos (second version;
 * DESIGN.md §8; the protocol is paper_1912_04232_b200/slabs.py).  A rank runs an ordinary md_system on a LOCAL
 * periodic box that holds its slab, copies of the neighbouring slabs' particles within r_cut + skin of it
 * (its halo) and an empty gap.  Local x = global x - T, except for the one periodic image the first and the
 * last rank take through the box boundary; every such translation is exact in fp32 (L72: the space is a
 * torus, a frame is a choice of origin), so pair displacements in a local frame are bit-identical to the
 * global ones.  The calls below are the coordinate plumbing of that scheme; the frame is plain data the
 * caller computes once (slabs.frames).
 *   kind 0 (first rank):  local = x, or (x - L) + Lx for x >= g2l_thr (the image of x near L);
 *                         global = local, or (local - Lx) + L for local >= l2g_thr
 *   kind 1 (middle):      local = x - T;  global = local + T
 *   kind 2 (last rank):   local = x for x < g2l_thr (the image of x near 0, raw), else x - T  (Lx = L - T);
 *                         global = local for local < l2g_thr, else local + T
 * A global x that rounds to >= L becomes 0.
 */
typedef struct md_slab_frame {
    int   kind;       /* 0 first, 1 middle, 2 last */
    float T;          /* translation (a multiple of 2^-8, >= 0) */
    float Lx;         /* local box side in x */
    float L;          /* global box side in x */
    float g2l_thr;    /* global x at which the image branch starts (kind 0) / ends (kind 2) */
    float l2g_thr;    /* local x at which the image zone starts (kind 0) / ends (kind 2) */
} md_slab_frame;

/* The opening of a step (v += dt/2m F, r = mu(r, dt v)) on the whole local system with every x put back on the
 * GLOBAL fp32 grid (x = to_local(to_global(x))): the rounding the global coordinate would get, so that a
 * decomposed run differs from md_nve_step only in the order forces are summed.  *flag is RAISED (never
 * cleared: several ranks of one process may share the word) when a particle is more than skin / 2 from where
 * the lists were built.  Halo copies (id[i] < 0) are left alone: their positions arrive from their owners.
 * stop (may be NULL): while *stop != 0 the call changes nothing.
 *
 * md_slab_force_half_kick: md_force_half_kick that changes nothing while *flag != 0 and then raises *stop;
 * *done (may be NULL) counts the calls that did run.  With these two the host can enqueue several steps
 * (drift, exchange, force) without waiting: from the first step whose drift meets a stale list on ANY rank
 * (the ranks share *flag, or all-reduce it between the two calls) every later call is a no-op, and the host
 * reads *done once per batch, rebuilds, and finishes the interrupted step with md_force_half_kick. */
int md_slab_kick_drift(md_system *sys, const md_slab_frame *frame, void *pos, void *vel, const void *force,
                       const int32_t *id, float dt, float mass, int32_t *flag, const int32_t *stop, void *stream);
int md_slab_force_half_kick(md_system *sys, const md_potential *pot, const void *pos, const int32_t *nbr_idx,
                            const int32_t *nbr_count, void *force, void *vel, float dt, float mass,
                            const int32_t *flag, int32_t *stop, int32_t *done, void *stream);

/* In place on the x component of n float4 positions: to_local != 0: global -> local, else local -> global. */
int md_slab_convert(const md_slab_frame *frame, void *pos, int n, int to_local, void *stream);

/* rows_out[k] = pos[slots[k]] with x made global (what a rank sends: its border particles);
 * pos[slots[k]] = rows[k] with x made local (what it receives: its halo copies).  slots: DEVICE int32[k]. */
int md_slab_pack(const md_slab_frame *frame, const void *pos, const int32_t *slots, int k, void *rows_out,
                 void *stream);
int md_slab_unpack(const md_slab_frame *frame, const void *rows, const int32_t *slots, int k, void *pos,
                   void *stream);

/* One step of a slab rank in two calls with the exchange between them.
 * md_slab_step_open  = md_slab_kick_drift, then both messages packed as md_slab_pack does (one launch).
 * md_slab_step_close = both received messages unpacked as md_slab_unpack does (one launch), then
 *                      md_slab_force_half_kick. */
int md_slab_step_open(md_system *sys, const md_slab_frame *frame, void *pos, void *vel, const void *force,
                      const int32_t *id, float dt, float mass, int32_t *flag, const int32_t *stop,
                      const int32_t *border_prev, int k_prev, void *rows_prev, const int32_t *border_next,
                      int k_next, void *rows_next, void *stream);
int md_slab_step_close(md_system *sys, const md_slab_frame *frame, const md_potential *pot, const void *rows_prev,
                       const int32_t *halo_prev, int h_prev, const void *rows_next, const int32_t *halo_next,
                       int h_next, void *pos, const int32_t *nbr_idx, const int32_t *nbr_count, void *force,
                       void *vel, float dt, float mass, const int32_t *flag, int32_t *stop, int32_t *done,
                       void *stream);

/*
 * The rebuild of a slab rank in five device phases (migration folded into the rebuild); every
 * array is DEVICE memory, positions float4 with x GLOBAL in the owned / row arrays and LOCAL in pos, ids int32
 * global particle numbers.  The caller reads the small count arrays back to size its messages; nothing else of
 * the rebuild passes through the host.  The order of the compacted outputs is not specified (one atomic per
 * warp); the cell list's canonical order makes the local system independent of it.
 *
 * md_slab_split:  the owned particles (id >= 0) among the n local slots, x made global, split by the slab
 *   [lo, hi): stayers to own_pos / own_vel / own_id (room for n), the others to the rows of the previous or the
 *   next rank, whichever is nearer round the periodic box: rows float[.][8] = position | velocity, ids int32.
 *   counts int32[4] = {stayers, to previous, to next, rows dropped because cap_rows was too small}.
 * md_slab_append: m received migrants (rows, ids) join the owned arrays at [offset, offset + m); *errors is
 *   incremented for each one outside [lo, hi) (it crossed more than one slab between two rebuilds).
 * md_slab_border: the owned particles with x < lo_edge (copies for the previous rank) and x >= hi_edge (for the
 *   next): rows float4 (x global), ids; map_prev / map_next (int32[number of particles of the whole system],
 *   all -1 between rebuilds) receive each one's position in its message.  counts int32[3] = {for previous, for
 *   next, dropped}.
 * md_slab_load:   the local system in pos / vel / id: the n_own owned particles, then the h_prev copies received
 *   from the previous rank, then the h_next from the next (velocity 0, id = -1 - global id), x made local;
 *   map_halo[global id] = position of the copy among the received rows (previous first).
 * md_slab_plan:   after md_cell_list_build and md_neighbor_list_build of that system: nbr_count = 0 for the
 *   copies (they take no force and no energy); border_prev / border_next / halo_slots = the slot each border
 *   particle / copy has now, in message order: what md_slab_pack and md_slab_unpack move every step.  The three
 *   maps are -1 again afterwards.
 * Errors: MD_EINVAL (NULL, negative sizes, bad frame), MD_ECUDA.
 */
int md_slab_split(const md_slab_frame *frame, float lo, float hi, const void *pos, const void *vel,
                  const int32_t *id, int n, void *own_pos, void *own_vel, int32_t *own_id, void *prev_rows,
                  int32_t *prev_ids, void *next_rows, int32_t *next_ids, int cap_rows, int32_t *counts,
                  void *stream);
int md_slab_append(const void *rows, const int32_t *ids, int m, float lo, float hi, void *own_pos, void *own_vel,
                   int32_t *own_id, int offset, int32_t *errors, void *stream);
int md_slab_border(float lo_edge, float hi_edge, const void *own_pos, const int32_t *own_id, int n_own,
                   void *prev_rows, int32_t *prev_ids, void *next_rows, int32_t *next_ids, int cap_rows,
                   int32_t *map_prev, int32_t *map_next, int32_t *counts, void *stream);
int md_slab_load(const md_slab_frame *frame, const void *own_pos, const void *own_vel, const int32_t *own_id,
                 int n_own, const void *halo_prev_rows, const int32_t *halo_prev_ids, int h_prev,
                 const void *halo_next_rows, const int32_t *halo_next_ids, int h_next, void *pos, void *vel,
                 int32_t *id, int32_t *map_halo, void *stream);
int md_slab_plan(const int32_t *id, int n, int32_t *nbr_count, int32_t *map_prev, int32_t *map_next,
                 int32_t *map_halo, int32_t *border_prev, int32_t *border_next, int32_t *halo_slots, void *stream);

/* BKS-type potential (L104 "Buckingham / BKS" [71-73], named only; reading A27): per species
 * pair the exp-6 term A_ab exp(-B_ab r) - C_ab / r^6, plus the Coulomb interaction of the species' point
 * charges in its damped shifted-force form (energy and force both vanish at r_cut):
 *   u_C = k_e q_a q_b [erfc(a r)/r - erfc(a rc)/rc + (erfc(a rc)/rc^2 + 2a/sqrt(pi) exp(-a^2 rc^2)/rc)(r - rc)]
 * host float[nspecies * nspecies] A, B, C (row-major, A >= 0, B > 0, C >= 0), host float[nspecies] charge,
 * 1 <= nspecies <= 4, coulomb_alpha = a >= 0, k_e >= 0.  Used by MD_KIND_BKS: md_potential.r_cut is the one
 * truncation radius (<= the list r_cut), shift applies to the exp-6 term, epsilon / sigma / alpha are
 * ignored; the species of a particle is (int)pos.w.  fp64 pair chain. */
int md_set_species_bks(md_system *sys, int nspecies, const float *A, const float *B, const float *C,
                       const float *charge, float coulomb_alpha, float k_e);

/* Diagnostic counters since md_create (or the last reset): copies int32[8] to the DEVICE buffer
 * `out` on `stream`, then clears them if reset != 0.
 *   out[0] particles whose force the fp32 fast path handed to the fp64 re-evaluation
 *   out[1..7] reserved (0) */
int md_counters(md_system *sys, int32_t *out, int reset, void *stream);

/* Cells per side n_k = floor(L_k / R) (1 for unused dimensions) -> host int[3]. */
int md_num_cells(const md_system *sys, int *ncell);

/*
 * Layout of a neighbor list (host out-pointers).  The dense N x capacity list of L74 is stored
 * in tiles of `tile` consecutive particles, slot-major inside a tile, so that the 32 lanes of a
 * warp read slot k of 32 particles as one 128-byte row: entry (i, k) lives at
 *     nbr_idx[(i / tile) * tile_stride + (i % tile) * particle_stride + k * slot_stride]
 * (currently tile = 32, tile_stride = 32 * capacity, particle_stride = 1, slot_stride = 32) and
 * a list buffer holds `length` = ceil(n / tile) * tile_stride int32.
 */
int md_nbr_layout(const md_system *sys, long *tile, long *tile_stride, long *particle_stride,
                  long *slot_stride, long *length);

/*
 * Cell list (L84 "partition.cell_list ... places them into cells where each cell has size
 * sigma"): cell coordinate c_k = min(n_k-1, (int)(x_k * fl32(n_k/L_k))), linear index
 * (c_z n_y + c_y) n_x + c_x, counting sort by cell.
 *   cell_start int32[cells+1] out: slots [cell_start[c], cell_start[c+1]) belong to cell c
 *   perm       int32[n]       out: perm[s] = index (on entry) of the particle in slot s;
 *                                  inside a cell slots ascend by x, ties by id (by index if id =
 *                                  NULL); md_neighbor_list_build relies on this order
 *   resort = 1: pos, vel (may be NULL) and id (may be NULL) are permuted in place so that
 *               new[s] = old[perm[s]];  resort = 0: they are left untouched.
 */
int md_cell_list_build(md_system *sys, void *pos, void *vel, int32_t *id,
                       int32_t *cell_start, int32_t *perm, void *stream);

/*
 * The same cell list (L84; md_cell_list_build with resort = 0 and id = NULL) through an entry point that
 * allocates NOTHING and needs neither a md_system nor a workspace: for callers that cannot call cudaMalloc
 * (code under CUDA graph capture, tight serving loops, harnesses that forbid it).  The counting sort's
 * scratch (cell of every particle, arrival rank, unsorted slots, histogram) lives in a static __device__ array
 * inside the library image: 832 KB that every GPU which loads the library holds until the process exits.
 * That fixes the LIMIT: n <= MD_STATIC_MAX_N particles and at most MD_STATIC_MAX_CELLS cells (the cells of
 * cfg: floor(L_k / (r_cut + skin)) per side); beyond either the call returns MD_EINVAL and launches nothing.
 *   cfg        the geometry, as for md_create (capacity and resort are checked but not used)
 *   pos        DEVICE float4[n] in: coordinates in [0, L); untouched
 *   cell_start DEVICE int32[cells + 1] out;  perm DEVICE int32[n] out: as md_cell_list_build
 *   pos_sorted DEVICE float4[n] out: pos_sorted[s] = pos[perm[s]] (must not alias pos)
 * The device is the one `pos` lives on.  The call makes no cudaMalloc / cudaFree and calls no allocating
 * library routine; on its first use per device it resolves the array's address (cudaGetSymbolAddress), which
 * a caller that captures graphs should let happen once before capturing.  Every call on a device shares the
 * one array, and the array keeps the last call's contents (the call clears the part that must start at zero):
 * two calls whose kernels OVERLAP on the GPU (different streams without an ordering between them) race.
 * Calls on one stream, or ordered by events, are safe.  Errors: MD_EINVAL, MD_EBOX, MD_ECUDA.
 */
#define MD_STATIC_MAX_N     65536
#define MD_STATIC_MAX_CELLS 16384
int md_cell_list_static(const md_config *cfg, int n, const void *pos, int32_t *cell_start, int32_t *perm,
                        void *pos_sorted, void *stream);

/*
 * Neighbor list (L84-L88 partition.neighbor_list; dense N x capacity rows, L74): for every
 * i all j != i in the 3^dim adjacent cells with r2 < R^2 under the canonical fp32 predicate
 * (nearest-image displacement with the box side subtracted from the larger
 * coordinate first; r2 = fma(dz,dz, fma(dy,dy, dx*dx)); strict <).
 *   pos        as left by md_cell_list_build (same cell_start / perm)
 *   nbr_idx    int32[length] out (md_nbr_layout): row i holds min(count_i, capacity) neighbor
 *              indices (in the particle order of `pos`), then the pad value n up to capacity;
 *              order within a row is unspecified
 *   nbr_count  int32[n] out: TRUE count, may exceed capacity
 *   status     int32[2] out: {1 if any count > capacity else 0, max true count}; rows of an
 *              overflowed list are truncated and forces from it are invalid
 * Also snapshots pos inside the workspace as the reference for md_needs_rebuild.
 */
int md_neighbor_list_build(md_system *sys, const void *pos, const int32_t *cell_start,
                           const int32_t *perm, int32_t *nbr_idx, int32_t *nbr_count,
                           int32_t *status, void *stream);

/* Rebuild test (L49 "whenever a particle moves by more than the halo distance", read as
 * half the skin): *flag = 1 if max_i ||d(pos_i, ref_i)||^2 > (skin/2)^2 else 0,
 * ref = positions at the last md_neighbor_list_build, nearest-image displacement. */
int md_needs_rebuild(md_system *sys, const void *pos, int32_t *flag, void *stream);

/*
 * Pair energy and force over the list (L78 U = 1/2 sum_{i!=j} u; L80 smap.neighbors;
 * L104 force = -grad U, written in closed form):
 *   LJ   u = 4 eps[(s/r)^12 - (s/r)^6] - shift*u(r_cut), r < r_cut
 *   SOFT u = eps/2 (1 - r/d_ij)^2, r < d_ij = (pos_i.w + pos_j.w)/2; r = 0: eps/2, no force
 *   MORSE u = eps (1 - exp(-alpha (r - sigma)))^2 - eps - shift*u(r_cut), r < r_cut (fp64 chain)
 *   BUCKINGHAM u = eps exp(-alpha r) - sigma / r^6 - shift*u(r_cut), r < r_cut (fp64 chain)
 *   force        float4[n] out: (F_i, e_i)
 *   energy_total double* out (may be NULL): sum_i e_i accumulated in fp64
 *   nbr_idx / nbr_count  any list in the md_nbr_layout layout whose rows hold every pair
 *                        within the potential's range (entries beyond it contribute nothing)
 * Precision: SOFT, 2-D and fast32 = 0: pair terms evaluated and accumulated in fp64
 * from exact displacements; 3-D LJ, Morse, Buckingham (default): fp32 pair terms with a per-particle error estimate,
 * fp64 re-evaluation of every particle whose estimate exceeds 1/3 of the 1e-5 force tolerance or
 * that has a pair within 1e-5 r_cut^2 of the truncation radius.  Rounded to fp32 once, on store.
 */
int md_pair_energy_force(md_system *sys, const md_potential *pot, const void *pos,
                         const int32_t *nbr_idx, const int32_t *nbr_count, void *force,
                         double *energy_total, void *stream);

/*
 * nsteps of velocity-Verlet NVE (L100 simulate.nve; L78 m r'' = -grad U; L72 shift function):
 *   v += dt/(2m) F;  r = wrap(r + dt v);  [rebuild test; if it fires: cell list (+ re-sort)
 *   and neighbor list];  F = F(r);  v += dt/(2m) F
 * with the rebuild decision taken on the device.  `force` must hold F(pos) on entry (call
 * md_neighbor_list_build + md_pair_energy_force once first); nbr_idx / nbr_count must be the
 * list of that build.  On exit pos/vel/force are the state after nsteps in the CURRENT
 * particle order; id[s] (may be NULL) = original index of the particle in slot s.  force.w is
 * left 0: the step loop does not evaluate energies (call md_pair_energy_force for e_i and E).
 *   stats int32[4] out: {steps done, rebuilds, first step (0-based) whose rebuild
 *                        overflowed or -1, max neighbor count seen in rebuilds}
 * stats is reset at the start of every call.
 */
int md_nve_step(md_system *sys, const md_potential *pot, void *pos, void *vel, void *force,
                int32_t *id, int32_t *nbr_idx, int32_t *nbr_count, float dt, float mass,
                int nsteps, int32_t *stats, void *stream);

/*
 * nsteps of overdamped (Brownian) dynamics at temperature kT (L100), kT = 0 being
 * gradient descent (L100), around the same device-side rebuild / force sequence:
 *   r_i = wrap(r_i + (dt/gamma) F_i + sqrt(2 kT dt / gamma) xi_i);  [rebuild];  F = F(r)
 * xi_i: standard normals of a counter-based generator keyed by (seed, step0 + s, id[i], pair
 * index) -- splitmix64 finaliser, two 24-bit uniforms, Box-Muller -- so a run is reproducible and
 * independent of the particle order the re-sort leaves; id = NULL keys by slot (resort = 0 only).
 *   force   must hold F(pos) on entry, holds F of the final positions on exit; there are no
 *           velocities; lists and stats as in md_nve_step.  Runs as CUDA graphs of 8 steps (rebuild in an IF
 *           node) unless use_graph = 0.
 */
int md_brownian_step(md_system *sys, const md_potential *pot, void *pos, void *force, int32_t *id,
                     int32_t *nbr_idx, int32_t *nbr_count, float dt, float gamma, float kT,
                     uint32_t seed, uint32_t step0, int nsteps, int32_t *stats, void *stream);

/*
 * nsteps of Langevin dynamics at temperature kT (L100), BAOAB splitting:
 *   v += dt/(2m) F;  r += dt/2 v;  v = c1 v + c2 xi (c1 = exp(-gamma dt), c2 = sqrt(kT/m (1-c1^2)));
 *   r = wrap(r + dt/2 v);  [rebuild];  F = F(r);  v += dt/(2m) F
 * xi as in md_brownian_step (same generator, keyed by seed, step0 + s, id[i]).  gamma = 0 is
 * md_nve_step's velocity Verlet.  force must hold F(pos) on entry; lists and stats as in md_nve_step.
 * CUDA graphs of 8 steps unless use_graph = 0.
 */
int md_langevin_step(md_system *sys, const md_potential *pot, void *pos, void *vel, void *force,
                     int32_t *id, int32_t *nbr_idx, int32_t *nbr_count, float dt, float mass,
                     float gamma, float kT, uint32_t seed, uint32_t step0, int nsteps, int32_t *stats,
                     void *stream);

/*
 * nsteps of NVT by a Nose-Hoover chain of M thermostats (L100 [67] Martyna, Klein and
 * Tuckerman's chains; M = option "nh_chain", default 1) around the velocity-Verlet step, explicit reversible
 * splitting; dof = dim n, Q_1 = dof kT tau^2, Q_j = kT tau^2 (j >= 2):
 *   T(dt);  v += dt/(2m) F;  r = wrap(r + dt v);  [rebuild];  F = F(r);  v += dt/(2m) F;  T(dt)
 *   T(dt), d = dt/2: K2 = sum m v^2; G_1 = (K2 - dof kT)/Q_1, G_j = (Q_{j-1} v_{j-1}^2 - kT)/Q_j;
 *          v_M += d/2 G_M; for j = M-1..1: a = exp(-d/4 v_{j+1}), v_j = (v_j a + d/2 G_j) a;
 *          v *= exp(-d v_1); K2 *= exp(-2d v_1); xi_j += d v_j; then j = 1..M-1 likewise and v_M += d/2 G_M
 *   nh_state  device double[2M] in/out = {xi_1..xi_M, v_1..v_M} (zero to start);
 *             H' = K + U + sum_j Q_j v_j^2/2 + dof kT xi_1 + kT sum_{j>=2} xi_j is the conserved quantity
 * force must hold F(pos) on entry; lists and stats as in md_nve_step.  CUDA graphs of 8 steps unless
 * use_graph = 0.
 */
int md_nose_hoover_step(md_system *sys, const md_potential *pot, void *pos, void *vel, void *force,
                        int32_t *id, int32_t *nbr_idx, int32_t *nbr_count, float dt, float mass,
                        float kT, float tau, double *nh_state, int nsteps, int32_t *stats, void *stream);

/* Flocking as an energy model (App. B, eqs. 3-10): ranges and strengths of
 * the alignment, avoidance and cohesion terms, the exponent of the cutoff function rho (eq. 6) and
 * the swimming speed v of eq. 4. */
typedef struct md_flock_params {
    float J_align, R_align;        /* eq. 7 (stop-gradient on the displacement: no position gradient) */
    float J_avoid, R_avoid;        /* eq. 8 */
    float J_cohesion, R_cohesion;  /* eqs. 9-10, D_i = sum over r < R_cohesion of (R_j - R_i) */
    float alpha;                   /* rho(r; Rc) = (1/alpha)(1 - r/Rc)^alpha, alpha >= 1 */
    float speed;                   /* v */
} md_flock_params;

/*
 * Disk obstacles of the boids model (App. B.3.1, eq. 11; reading A26):
 *   e_io = J rho(r_io; D_o) (1 + N_i . Rhat_io)^2,  R_io = C_o - R_i (nearest image)
 * added to E in md_flock_step from the next call on (gradients in R_i and theta_i).
 *   nobs    0..MD_MAX_OBSTACLES (0 removes them)
 *   centre  HOST float[nobs*2], inside the box;  radius  HOST float[nobs], 0 < D_o < L/2;  J >= 0
 * The values are copied into the context; MD_EINVAL otherwise.
 */
#define MD_MAX_OBSTACLES 16
int md_flock_obstacles(md_system *sys, int nobs, const float *centre, const float *radius, float J);

/*
 * Predators of the boids model (App. B.3.2, eqs. 12-13; reading A28): a second,
 * small population with the same state.  Each side descends its own energy in its own coordinates:
 *   boids add      sum_p J_flee rho(r_ip; R_flee) (1 + N_i . Rhat_ip)^2   (the obstacle energy, predator = disk)
 *   predators use  1/2 J_chase (1 - Dhat_p . N_p)^2 + the obstacle term,  D_p = sum_{r_ip < R_chase} (R_i - R_p)
 * and move by forward Euler at their own speed, all from the state at the start of the step.
 *   npred  0..MD_MAX_PREDATORS (0 removes them)
 *   pred   DEVICE float4[npred] in/out: (x, y, 0, theta_p); owned by the caller, read and written by every
 *          md_flock_step until replaced; 16-byte aligned
 *   par    J >= 0, R_flee and R_chase in (0, L/2), speed >= 0 (copied)
 * The chase sum runs over all boids (one block per predator), not over the neighbor list.
 */
#define MD_MAX_PREDATORS 16
typedef struct md_predator_params {
    float J_flee, R_flee;      /* boids: eq. 12's boid-predator term */
    float J_chase, R_chase;    /* predators: eq. 13's predator-boid term */
    float speed;               /* predators' swimming speed */
} md_predator_params;
int md_flock_predators(md_system *sys, int npred, void *pred, const md_predator_params *par);

/*
 * nsteps of the boids model by forward Euler (eqs. 4-5) on a 2-D system:
 *   R_i' = wrap(R_i + dt (v N(theta_i) - grad_{R_i} E));  theta_i' = theta_i - dt grad_{theta_i} E
 * with E = E_align + E_avoid + E_cohesion over the neighbor list (every range <= the list r_cut) plus the
 * obstacle term of md_flock_obstacles and the predators of md_flock_predators, both
 * updates from the state at the start of the step; then the device-side rebuild test and rebuild.
 *   pos   float4[n] in/out: (x, y, 0, theta_i) -- the heading travels in pos.w
 *   lists, id and stats as in md_nve_step (the list must be valid for pos on entry)
 * CUDA graphs of 8 steps unless use_graph = 0.  fp64 accumulation over the list, fp32 state.
 */
int md_flock_step(md_system *sys, const md_flock_params *par, void *pos, int32_t *id, int32_t *nbr_idx,
                  int32_t *nbr_count, float dt, int nsteps, int32_t *stats, void *stream);

/* FIRE parameters (Bitzek et al. 2006; the paper names "FIRE Descent", L100, and uses it in §4.2). */
typedef struct md_fire_params {
    float dt_start, dt_max;   /* first step size; cap */
    int   n_min;              /* steps with P > 0 before dt grows */
    float f_inc, f_dec;       /* growth (>= 1) and cut (in (0,1)) of dt */
    float alpha_start;        /* mixing parameter after a reset, in [0,1) */
    float f_alpha;            /* its decay per growing step, in (0,1] */
} md_fire_params;

/*
 * nsteps of FIRE minimisation (L100, L322) with unit mass, around the same drift /
 * device-side rebuild / force sequence as md_nve_step:
 *   v += dt/2 F;  r = wrap(r + dt v);  [rebuild];  F = F(r);  v += dt/2 F;
 *   P = sum F.v:  P > 0: v = (1-alpha) v + alpha |v| F/|F|, n_pos += 1, and once n_pos > n_min
 *   dt = min(dt f_inc, dt_max), alpha *= f_alpha;  else v = 0, n_pos = 0, dt *= f_dec,
 *   alpha = alpha_start.
 *   fire_state  device float[4] in/out = {dt, alpha, n_pos, sign of the last P}; dt <= 0 on entry
 *               starts from (dt_start, alpha_start, 0); pass it back unchanged to continue a run
 *   force       must hold F(pos) on entry, holds F of the final positions on exit; the lists as in
 *               md_nve_step; stats as in md_nve_step.  CUDA graphs of 8 steps unless use_graph = 0.
 */
int md_fire_minimize(md_system *sys, const md_potential *pot, const md_fire_params *par, void *pos,
                     void *vel, void *force, int32_t *id, int32_t *nbr_idx, int32_t *nbr_count,
                     float *fire_state, int nsteps, int32_t *stats, void *stream);

/*
 * End-to-end convenience over HOST buffers: copies pos/vel in, builds the lists, evaluates F,
 * runs nsteps of md_nve_step and copies the state back un-permuted (original particle order).
 * Synchronous.  The device allocation, the system and its step graphs are kept for the next call
 * with the same (cfg, n, current device) -- one context per process, replaced when they differ,
 * dropped on any error and by md_nve_run_host_release(); calls are serialised by a mutex.
 *   pos_host, vel_host   host float4[n] in/out
 *   force_host           host float4[n] out (may be NULL)
 *   energy_host          host double out (may be NULL): potential energy of the final state
 *   stats_host           host int32[4] out (may be NULL)
 */
int md_nve_run_host(const md_config *cfg, const md_potential *pot, int n, void *pos_host,
                    void *vel_host, void *force_host, double *energy_host, float dt,
                    float mass, int nsteps, int32_t *stats_host);

/* Frees the context md_nve_run_host keeps between calls (no-op if there is none). */
int md_nve_run_host_release(void);

#ifdef __cplusplus
}
#endif
#endif /* MD_B200_H */
