// Internal declarations shared by the host set-up, the kernels and the C-ABI layer.
// Not installed; the public boundary is include/landau.h.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "landau.h"

namespace landau {

// Everything landau_create computes on the host ("assembled once
// on the CPU ... amortized").  Plain vectors; uploaded verbatim.
struct HostSpace {
    int p = 0, Nq = 0, Nb = 0;
    int64_t Ne = 0, N = 0, n = 0, nnz = 0;
    std::vector<double> r, z, w_in, w_out;   // [N]
    std::vector<double> invJ;                // [Ne][2]  (2/hr, 2/hz)
    std::vector<double> B, E0, E1;           // [Nq][Nb] psi_a(x_q), d/dxi psi_a, d/deta psi_a
    std::vector<int32_t> lptr, ldof;         // local node (e*Nb+a) -> free DOFs (CSR)
    std::vector<double> lw;                  //                     ... and weights
    std::vector<double> dof_r, dof_z;        // [n]
    std::vector<int32_t> rowptr, colidx;     // A1 pattern
    std::vector<int32_t> gptr, gidx;         // nnz k -> entries e*Nb*Nb + a*Nb + b of C_e
    std::vector<double> gw;                  //          ... with weight P_e[a,row] P_e[b,col]
    std::vector<int32_t> cptr, cidx;         // dof d -> entries e*Nb + a of the element vectors
    std::vector<double> cw;
};

// Returns LANDAU_OK or LANDAU_EINVAL (message in err).
int build_host_space(const landau_mesh &mesh, int order, HostSpace &hs, std::string &err);

}  // namespace landau
