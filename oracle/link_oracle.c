/*
 * ORACLE for the linking step (test infrastructure only -- never linked into or imported by the product path).
 *
 * Plain, single-threaded C restatement of "pairwise relations" (Sec. 2.2 and 2.2.2): the
 * elements are already sorted by time, so an element with a larger index never precedes one with a smaller
 * index; for every pair i<j the two elements are related iff they are timelike separated; the
 * result is the dense N x N binary adjacency matrix, symmetric, no self loops.
 * Output here is one byte per entry (B[i*N+j] in {0,1}); packing is the caller's business.
 *
 * Timelike-separation tests, all in double with one rounding per operation (compile with
 * -ffp-contract=off so no FMA is formed):
 *   geometry 0  (1+1) Minkowski diamond in light-cone coordinates (u,v):   u_i < u_j and v_i < v_j
 *               [NOT IN PAPER: BASELINE.json configs 0,1,4; reading A17]
 *   geometry 1  (3+1) Minkowski (t,x,y,z):   dt > 0 and dt*dt > (dx*dx + dy*dy) + dz*dz
 *               [NOT IN PAPER: BASELINE.json configs 2,3; reading A17]
 *   geometry 2  (1+1) de Sitter, conformal time eta and angle theta (Sec. 5.1, below Eq. 9):
 *               "pi - |pi - |theta_1 - theta_2|| < |eta_1 - eta_2|"; direction from the index order.
 *
 * Parity pins (tests/test_link_pins.py): 2D relations = C(N,2) - inversions (merge sort on ranks); 4D
 * ordering fraction -> Gamma(5)Gamma(2)/(2 Gamma(6)) = 1/10 over seeds; de Sitter ordering fraction =
 * E|eta_1-eta_2|/pi by quadrature; hand-placed events on / inside / outside the light cone; chains and
 * antichains; transitivity, symmetry and zero diagonal of every result.
 */
#include <math.h>
#include <stdint.h>
#include <string.h>

#define LINK_PI 3.14159265358979323846

/* Is element a (smaller index, not later in time) related to element b?  ca, cb: their coordinates. */
static int timelike(int geometry, const double *ca, const double *cb)
{
    if (geometry == 0) {
        return ca[0] < cb[0] && ca[1] < cb[1];
    } else if (geometry == 1) {
        double dt = cb[0] - ca[0], dx = cb[1] - ca[1], dy = cb[2] - ca[2], dz = cb[3] - ca[3];
        double s2 = dx * dx + dy * dy;
        s2 = s2 + dz * dz;
        return dt > 0.0 && dt * dt > s2;
    } else {
        double dth = fabs(ca[1] - cb[1]);
        double lhs = LINK_PI - fabs(LINK_PI - dth);
        double rhs = fabs(ca[0] - cb[0]);
        return lhs < rhs;
    }
}

int csg_oracle_link_dim(int geometry) { return geometry == 1 ? 4 : 2; }

/* coords: N x dim doubles, row per element, sorted by time.  B: N*N bytes, overwritten. */
void csg_oracle_link(int geometry, const double *coords, int64_t N, uint8_t *B)
{
    const int dim = csg_oracle_link_dim(geometry);
    memset(B, 0, (size_t)N * (size_t)N);
    for (int64_t i = 0; i < N; ++i)
        for (int64_t j = i + 1; j < N; ++j)
            if (timelike(geometry, coords + dim * i, coords + dim * j)) {
                B[i * N + j] = 1;   /* i precedes j */
                B[j * N + i] = 1;   /* undirected storage: the matrix is symmetric */
            }
}
