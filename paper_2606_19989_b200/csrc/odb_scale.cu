// Loss-scaling weights per slot: section 2.3 "Loss scaling" Eq. 2, the
// sample-level rule P:65, approximate vs exact mode App. B, the three modes P:738.
// fp64 throughout; every arithmetic step is ONE correctly rounded IEEE operation (__ddiv_rn,
// __dmul_rn, __dadd_rn: no contraction into FMA), sums over ranks run in the order r = 0..R-1, so the
// result is bit-identical to a sequential CPU evaluation of the same formulas.  sm_100a only.
#include "odb_internal.cuh"

namespace odb {

// pass 1, one thread per slot: the numerator of w_{r,k}
//   SAMPLE: n;  TOKEN_EXACT: t (post-alignment valid tokens);
//   TOKEN_APPROX: n * (t_orig / n_orig) over the slots of the same rank cut from the same candidate
//   group -- a run of consecutive steps that starts at the head slot grp_origin[s] (U27).
__global__ void k_loss_num(int mode, int R, int n_steps, const int32_t *__restrict__ grp_count,
                           const int32_t *__restrict__ grp_valid, const int32_t *__restrict__ grp_origin,
                           double *__restrict__ w) {
    const int64_t n_slots = (int64_t)R * n_steps;
    for (int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; s < n_slots; s += (int64_t)gridDim.x * blockDim.x) {
        double num;
        if (mode == ODB_SCALE_SAMPLE) {
            num = (double)grp_count[s];
        } else if (mode == ODB_SCALE_TOKEN_EXACT) {
            num = (double)grp_valid[s];
        } else {
            const int r = (int)(s / n_steps);
            const int64_t row = (int64_t)r * n_steps;
            const int o = grp_origin[s];
            long long t_orig = 0, n_orig = 0;
            for (int k = o; k < n_steps && grp_origin[row + k] == o; ++k) {
                t_orig += grp_valid[row + k];
                n_orig += grp_count[row + k];
            }
            const double tbar = n_orig > 0 ? __ddiv_rn((double)t_orig, (double)n_orig) : 0.0;
            num = __dmul_rn((double)grp_count[s], tbar);
        }
        w[s] = num;
    }
}

// pass 2, one thread per step: denominator = sum over ALL ranks of the job in rank order, then the
// quotients of the local ranks.  num_world is rank-major [world_ranks][n_steps]; the local ranks are
// rows [rank_offset, rank_offset + R).  w may alias the local rows of num_world.
__global__ void k_loss_norm(int R, int world_ranks, int rank_offset, int n_steps, const double *num_world, double *w) {
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < n_steps; k += gridDim.x * blockDim.x) {
        double denom = 0.0;
        for (int q = 0; q < world_ranks; ++q) denom = __dadd_rn(denom, num_world[(int64_t)q * n_steps + k]);
        for (int r = 0; r < R; ++r) {
            const double num = num_world[(int64_t)(rank_offset + r) * n_steps + k];
            w[(int64_t)r * n_steps + k] = denom > 0.0 ? __ddiv_rn(num, denom) : 0.0;
        }
    }
}

cudaError_t launch_loss_numerators(odb_ctx *c, int mode, double *d_num, cudaStream_t st) {
    const int R = c->prm.n_ranks, n_steps = c->n_steps;
    const int64_t n_slots = (int64_t)R * n_steps;
    if (n_slots == 0) return cudaSuccess;
    const int blocks = (int)std::min<int64_t>((n_slots + 255) / 256, (int64_t)c->sm_count * 8);
    k_loss_num<<<blocks, 256, 0, st>>>(mode, R, n_steps, c->grp_count.p, c->grp_valid.p, c->grp_origin.p, d_num);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_loss_normalize(odb_ctx *c, const double *d_num_world, int world_ranks, int rank_offset,
                                  double *d_weights, cudaStream_t st) {
    const int R = c->prm.n_ranks, n_steps = c->n_steps;
    if ((int64_t)R * n_steps == 0) return cudaSuccess;
    const int blocks = (int)std::min<int64_t>(((int64_t)n_steps + 127) / 128, (int64_t)c->sm_count * 8);
    k_loss_norm<<<blocks, 128, 0, st>>>(R, world_ranks, rank_offset, n_steps, d_num_world, d_weights);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_loss_weights(odb_ctx *c, int mode, double *d_weights, cudaStream_t st) {
    cudaError_t e = launch_loss_numerators(c, mode, d_weights, st);
    if (e != cudaSuccess) return e;
    return launch_loss_normalize(c, d_weights, c->prm.n_ranks, 0, d_weights, st);  // in place: world = local
}

}  // namespace odb
