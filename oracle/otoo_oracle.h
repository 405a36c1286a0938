/* otoo_oracle.h -- plain, slow, fp64 CPU oracle for the OTOO force path (arxiv 1206.1199).
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing in the product path (paper_1206_1199_b200/, include/)
 * may include, link or call this; only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs do.  It shares no code with the CUDA path.
 *
 * The method is an approximation (a tree code), so the oracle follows the algorithm step by
 * step in the paper's order (section II, III-B, III-C, III-D), with the readings
 * R1..R24 listed in DESIGN.md.  The O(N^2) definition (orc_direct_sum) is its truth check.
 * All host pointers.  Positions/masses come in as fp32 (single precision),
 * every sum is fp64; the quantities that decide an integer (key quantisation, the MAC compare,
 * the SPH neighbour compare) are evaluated in fp32 exactly as DESIGN.md states.
 *
 * Pins (tests/test_oracle_*.py, tests/test_golden.py): brute-force octants, stable sort, tree invariants, two-particle
 * cell, r_b = l/theta + s on a three-particle tree done by hand, tiling invariant of the lists, stackless
 * walk == recursive walk, theta=0 == direct sum, Newton's third law, two-body closed form, Plummer
 * potential, kernel normalisation, lattice density, brute-force SPH neighbour sets; the abs_sum outputs (the
 * denominators of the GPU parity tolerance) against numpy sums over the exported lists / all pairs, one-pair closed
 * forms and |sum| <= sum of magnitudes; Delta-MAC: two-particle cell and Eq. 3, B2 bottom-up == Eq. 2
 * direct, per-cell error <= Delta, r_b limits (L81), measured Delta exponents at n_vec = 4 / 8; group distance from
 * the pieces' boxes (R25, default) and the exact minimum (L163; R23): brute force over pieces / members with the
 * pieces recomputed from the exported keys, lists nested exact <= pieces <= one box; SPH walk per piece (R26): same
 * neighbours, brute-force supersets; Hilbert keys (L131): bijection, face adjacency of consecutive keys, hierarchy,
 * inverse, same cells as the Morton tree; adaptive h: fixed point, lattice count steps; div v / rot v: linear
 * fields, rigid rotation; artificial viscosity: alpha = 0 / f = 0 limits, receding flow, momentum and energy
 * balance, two-particle closed form.
 * The absolute accuracy of the theta-MAC has no figure in PAPER.md (its error plot, Fig. 5, is for the Delta-MAC and is
 * missing); it is pinned to the multipole remainder instead (test_theta_mac_error_is_bounded_by_the_multipole_remainder:
 * every target outside r_b of every accepted cell, |a_exact - a_monopole| <= 3 M b^2 / (d - b)^4 per (target, cell) by
 * brute force, the walk's force within the sum of these remainders of the O(N^2) sum, median error ~ theta^2.4).
 */
#ifndef OTOO_ORACLE_H
#define OTOO_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct orc_tree orc_tree;

typedef struct {
  uint64_t prefix;      /* key >> 3*(21-level) */
  uint32_t first;       /* first sorted slot */
  uint32_t count;       /* particles in the cell */
  uint32_t child_first; /* canonical id of first child, 0 if leaf */
  uint8_t level;        /* 0 = root */
  uint8_t child_count;  /* 0 if leaf */
} orc_cell;

/* O(N^2) softened Plummer direct sum (fp64).  acc_pot[4*t..] = (ax,ay,az,phi) of target
 * index targets[t] (targets==NULL: all N in order, n_targets ignored). */
void orc_direct_sum(int64_t N, const float* pos_mass, double eps, int64_t n_targets,
                    const int64_t* targets, double* acc_pot);

/* Tree build: PAPER.md III-B steps 1-4 + III-C (mass, centre of mass). */
orc_tree* orc_build(int64_t N, const float* pos_mass, int n_crit);
/* key_order 0: Morton keys (R3); 1: Hilbert keys (reading R20: Skilling's transpose form) */
orc_tree* orc_build_ord(int64_t N, const float* pos_mass, int n_crit, int key_order);
uint64_t orc_hilbert_key(const uint32_t q[3]);           /* 21-bit coordinates -> 63-bit Hilbert key */
void orc_hilbert_coords(uint64_t key, uint32_t q[3]);    /* and back */
void orc_free(orc_tree*);
int64_t orc_ncell(const orc_tree*);
int64_t orc_nleaf(const orc_tree*);
int orc_depth(const orc_tree*);
void orc_root(const orc_tree*, float lo[3], float* S);
/* canonical order (level asc, first asc). Any pointer may be NULL. */
void orc_export(const orc_tree*, uint32_t* perm, uint64_t* keys, orc_cell* cells,
                float* cell_com_m /*4*ncell*/, double* cell_s /*ncell*/,
                double* cell_M_P /*4*ncell: M, Px, Py, Pz*/);
/* key of a single point for the tree's root cube (R2, R3). */
uint64_t orc_key(const orc_tree*, const float xyz[3]);

/* rb^2 (fp32) for each cell under the theta-MAC.  mac_kind 0: r_b = l/theta + s (default),
 * 1: r_b = l/theta. */
void orc_rb2(const orc_tree*, double theta, int mac_kind, float* rb2 /*ncell*/);

/* The paper's absolute-error MAC (Eq. 1-2; reading R19 for the summation order of B2).
 * B2, bmax: ncell doubles each (bmax may be NULL). */
void orc_delta_cell_props(const orc_tree*, double* B2, double* bmax);
double orc_B2_direct(const orc_tree*, int64_t cell);      /* Eq. 2 written out, for the pin */
void orc_rb2_delta(const orc_tree*, double delta, double m_limit, float* rb2 /*ncell*/);
/* Group walk + gravity sums with a given rb^2 per cell (any MAC of the form "accept iff d > r_b", L61). */
uint64_t orc_gravity_rb2(const orc_tree*, double eps, const float* rb2, int group_size, int walk_kind,
                         const int64_t* sel, int64_t nsel, double* acc_pot, uint32_t* n_tests,
                         uint32_t* n_cells, uint32_t* n_parts, double* abs_sum);

/* Group walk + gravity sums.  Outputs in the CALLER's original particle order.
 * walk_kind 0: recursive (R9); 1: stackless next/more exactly as PAPER.md L57.
 * group counters are per group g = sorted slots [gG, min((g+1)G, N)). Pointers may be NULL
 * (acc_pot NULL = count only). Returns total interactions (R11). */
uint64_t orc_gravity(const orc_tree*, double eps, double theta, int group_size, int mac_kind,
                     int walk_kind, double* acc_pot /*4N*/, uint32_t* n_tests, uint32_t* n_cells,
                     uint32_t* n_parts, double* abs_sum /*N or NULL: sum_j |a_ij| over the same lists*/);
/* The same for a selection of groups only (sel[0..nsel) group indices; counters indexed by position
 * in sel; acc_pot/abs_sum still 4N/N, written for the selected groups' targets only). */
uint64_t orc_gravity_sel(const orc_tree*, double eps, double theta, int group_size, int mac_kind,
                         int walk_kind, const int64_t* sel, int64_t nsel, double* acc_pot,
                         uint32_t* n_tests, uint32_t* n_cells, uint32_t* n_parts, double* abs_sum);
/* the lists of one group (sizes from orc_gravity counters) */
void orc_group_lists(const orc_tree*, double theta, int group_size, int mac_kind, int64_t g,
                     uint32_t* cell_ids, uint32_t* part_slots);

void orc_group_lists_rb2(const orc_tree*, const float* rb2, int group_size, int64_t g,
                         uint32_t* cell_ids, uint32_t* part_slots);

/* SPH.  h = support radius per particle (original order).  */
void orc_sph_cell_radii(const orc_tree*, const float* h, float* bmax, float* rsph /*ncell each*/);
uint64_t orc_sph_density(const orc_tree*, const float* h, int group_size, double* rho,
                         uint32_t* nngb, uint32_t* n_tests, uint32_t* n_parts);
uint64_t orc_sph_density_sel(const orc_tree*, const float* h, int group_size, const int64_t* sel,
                             int64_t nsel, double* rho, uint32_t* nngb, uint32_t* n_tests, uint32_t* n_parts);
/* SPH stage 1 with velocity derivatives (PAPER L252 step 4; reading R22): out = 4N (div v, rot v), rho = N or NULL */
uint64_t orc_sph_divrot_sel(const orc_tree*, const float* h, const float* vel /*4N*/, int group_size,
                            const int64_t* sel, int64_t nsel, double* rho, double* out, double* abs_sum);
/* adaptive h (reading R21): iterate h in place towards n_target neighbours (+- tol); returns iterations */
int orc_sph_adapt_h(const orc_tree*, float* h, double n_target, double tol, int max_iter, int group_size,
                    uint32_t* nngb_out);
/* candidate list of one SPH group (sorted slots) */
void orc_sph_group_list(const orc_tree*, const float* h, int group_size, int64_t g,
                        uint32_t* part_slots);
uint64_t orc_sph_force(const orc_tree*, const float* h, const double* rho, const double* P,
                       const float* vel /*4N or NULL*/, int group_size, double* acc_dudt /*4N*/,
                       double* abs_sum /*2N or NULL: sum_j |a_ij|, sum_j |du_ij|*/);
uint64_t orc_sph_force_sel(const orc_tree*, const float* h, const double* rho, const double* P,
                           const float* vel, int group_size, const int64_t* sel, int64_t nsel,
                           double* acc_dudt, double* abs_sum);
/* the same with artificial viscosity (reading R24): visc = 4N floats (c, alpha, Balsara f, -), vel required */
uint64_t orc_sph_force_visc_sel(const orc_tree*, const float* h, const double* rho, const double* P,
                                const float* vel, const float* visc, int group_size, const int64_t* sel,
                                int64_t nsel, double* acc_dudt, double* abs_sum);
/* cubic spline with support h (R13) */
double orc_W(double r, double h);
double orc_dWdr(double r, double h);

/* group-cell distance: 2 (default) = minimum over the tight boxes of the group's pieces between its 7 coarsest key
 * boundaries (R25; the SPH walks apply their test per piece with the piece's own h_max, R26); 0 = from one box per
 * group (R8 / R15); 1 = the paper's exact minimum over the group's members (R23; SPH walks: one box). */
void orc_set_dist_kind(orc_tree*, int kind);
void orc_set_split_pieces(orc_tree*, int K);   /* dist_kind 2: pieces per group (8 = the reading R25; other values for the study in DESIGN.md only) */
int orc_max_threads(void);
void orc_set_threads(int n);
#ifdef __cplusplus
}
#endif
#endif
