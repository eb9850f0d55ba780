// Balloon-Windkessel BOLD read-out per region (Extended Data Table 4; reading R30 in DESIGN.md):
//   s' = z - kappa s - gamma (f - 1),  f' = s,  tau v' = f - v^(1/alpha),
//   tau q' = f E(f, rho) / rho - v^(1/alpha) q / v,  E = 1 - (1 - rho)^(1/f),
//   y = V0 [k1 (1 - q) + k2 (1 - q / v) + k3 (1 - v)],
// one explicit Euler step ("the Euler-Maruyama discrete-time version"; no noise term) per completed
// region-rate window, z = z_scale * region rate in Hz ("the spike rate of a pool of neurons").
//
// Off the step loop: the region-count windows are kept as a history ring (a4), so the model catches up after a
// batch of steps -- one thread per region walks the windows it has not consumed yet.  fp64; the operation order
// is the one written here (the library is built with -fmad=false).
#include "db_host.h"

namespace dbk {

__global__ void __launch_bounds__(128) k_bold(const __grid_constant__ SimDev p, const BoldDev b) {
    const int r = (int)(blockIdx.x * blockDim.x + threadIdx.x);
    if (r >= p.n_regions) return;
    const unsigned long long done = p.ctl->step / (unsigned long long)p.window_steps;   // completed windows
    double s = b.state[4 * r + 0], f = b.state[4 * r + 1], v = b.state[4 * r + 2], q = b.state[4 * r + 3];
    const double sc = b.scale[r];                    // z_scale / (region size * window seconds)
    const double inv_alpha = 1.0 / b.alpha, om_rho = 1.0 - b.rho;
    for (unsigned long long w = *b.cursor; w < done; ++w) {
        const double z = (double)p.region_counts[(size_t)(w % p.max_windows) * p.n_regions + r] * sc;
        const double fout = pow(v, inv_alpha);
        const double E = 1.0 - pow(om_rho, 1.0 / f);
        const double ds = (z - b.kappa * s) - b.gamma * (f - 1.0);
        const double df = s;
        const double dv = (f - fout) / b.tau;
        const double dq = ((f * E) / b.rho - (fout * q) / v) / b.tau;
        s = s + b.h * ds; f = f + b.h * df; v = v + b.h * dv; q = q + b.h * dq;
    }
    b.state[4 * r + 0] = s; b.state[4 * r + 1] = f; b.state[4 * r + 2] = v; b.state[4 * r + 3] = q;
    b.y[r] = b.V0 * ((b.k1 * (1.0 - q) + b.k2 * (1.0 - q / v)) + b.k3 * (1.0 - v));
}

__global__ void k_bold_advance(const __grid_constant__ SimDev p, const BoldDev b) {
    *b.cursor = p.ctl->step / (unsigned long long)p.window_steps;
}

__global__ void k_bold_init(const BoldDev b, const int n_regions) {
    const int r = (int)(blockIdx.x * blockDim.x + threadIdx.x);
    if (r == 0) *b.cursor = 0ull;
    if (r >= n_regions) return;
    b.state[4 * r + 0] = 0.0; b.state[4 * r + 1] = 1.0; b.state[4 * r + 2] = 1.0; b.state[4 * r + 3] = 1.0;   // rest
    b.y[r] = 0.0;
}

cudaError_t launch_bold_init(const BoldDev& b, int n_regions, cudaStream_t st) {
    k_bold_init<<<(n_regions + 127) / 128, 128, 0, st>>>(b, n_regions);
    return cudaGetLastError();
}

// Consume every completed window since the last call (the caller keeps the batches shorter than the history ring).
cudaError_t launch_bold(const SimDev& p, const BoldDev& b, cudaStream_t st) {
    k_bold<<<(p.n_regions + 127) / 128, 128, 0, st>>>(p, b);
    k_bold_advance<<<1, 1, 0, st>>>(p, b);
    return cudaGetLastError();
}

}  // namespace dbk
