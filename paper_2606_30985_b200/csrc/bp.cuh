// bp.cuh - BP sweep / Bethe / field-gate launchers (see bp.cu).
#pragma once
#include "common.cuh"

namespace pepo {

#define PEPO_BP_MAXS 32
#define PEPO_BP_MAXCHUNK 32

struct BpSite {
  const double* T;            // pinned slab psi_v[..., p_v], dims d[0..3] = (U,D,L,R), 1 if absent
  int d[4];
  int present[4];
  int first_slot;             // first present leg (site value vs_v is taken there)
  const double* in[4];        // incoming message per slot (a constant [1.0] if absent)
  const double* out_old[4];   // current outgoing message per slot
  double* out_new[4];         // next outgoing message per slot
  double* partU; double* partD; double* partS;   // partU/partD: one row per chunk of (l,r) slices
  int chunk, nchunks;         // (l,r) slices per CTA of bp_partial_kernel, CTAs for this site
  double* vs;                 // site scalar of eq. (7)
};
struct BpBatch {
  int count; BpSite s[PEPO_BP_MAXS];
  // grouped sweeps: if skip_if != nullptr and the delta stored there (bit pattern of a non-negative
  // double, written by the previous sweep of the group) is below skip_tol, the kernels of this sweep
  // return at once: the previous sweep had converged (eq. (14)); a skipped sweep leaves its own
  // delta slot at 0, so every later sweep of the group is skipped too
  const unsigned long long* skip_if = nullptr;
  double skip_tol = 0.0;
};

struct FieldBatch {
  int count;
  double* psi[PEPO_BP_MAXS];
  long long slab[PEPO_BP_MAXS];
  double G[16];
  int row_mask, col_mask;
};

int launch_bp_partial(cudaStream_t st, const BpBatch& b);
int launch_bp_finalize(cudaStream_t st, const BpBatch& b, double damping, int update,
                       unsigned long long* delta_bits, int* flag);
int launch_bp_init(cudaStream_t st, double* msgs, const int* chi_of_msg, int n_msgs, int chi_max, int mode);
int launch_bethe(cudaStream_t st, const double* vs, int n_sites, const double* msgs,
                 const int* chi_of_msg, int n_bonds, int chi_max, double* out_C, int* out_status);
int launch_field_gate(cudaStream_t st, const FieldBatch& b);
// Per-site Pauli-resolved norms (n(r,t) of PAPER.md section 6.4): w[site][p] = sum_i psi[i,p]^2 prod_legs
// lambda_leg[i_leg]; one pass over the four slabs of every site, per-chunk partials summed in fixed order.
#define PEPO_SW_CHUNKS 64
struct SiteWeightBatch {
  int count;
  const double* psi[PEPO_BP_MAXS];
  int d[PEPO_BP_MAXS][4];                 // leg dims in storage order (1 if absent)
  const double* lam[PEPO_BP_MAXS][4];     // lambda of the leg's bond (a constant [1.0] if absent)
  double* part[PEPO_BP_MAXS];             // PEPO_SW_CHUNKS x 4 partials
  double* out[PEPO_BP_MAXS];              // 4 doubles: w_I, w_X, w_Y, w_Z
};
int launch_site_weights(cudaStream_t st, const SiteWeightBatch& b);
int launch_bond_entropy(cudaStream_t st, const double* lambda, const int* chi_of_msg, int n_bonds, int chi_max,
                        double* out);

}  // namespace pepo
