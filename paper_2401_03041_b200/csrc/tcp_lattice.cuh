// Lattice tables (App. B) as compile-time functions.
//
// D3Q27 is indexed as a tensor product: q = 9*(cz+1) + 3*(cy+1) + (cx+1), q = 13 is the rest
// velocity and the opposite of q is 26 - q.  The smaller thermal stencils keep the velocities
// whose |c|^2 class the stencil has, in ascending q order (so the opposite of compact index k is
// Q-1-k).  Weights: eqs. B.1-B.4.
#pragma once
#include <type_traits>
#include <utility>

namespace tcp {

__host__ __device__ constexpr int q27(int cx, int cy, int cz) { return 9 * (cz + 1) + 3 * (cy + 1) + (cx + 1); }
__host__ __device__ constexpr int cx27(int q) { return q % 3 - 1; }
__host__ __device__ constexpr int cy27(int q) { return (q / 3) % 3 - 1; }
__host__ __device__ constexpr int cz27(int q) { return q / 9 - 1; }
__host__ __device__ constexpr int cls27(int q) {
    return cx27(q) * cx27(q) + cy27(q) * cy27(q) + cz27(q) * cz27(q);
}

// does stencil Q contain velocity class c2 = |c|^2 ?
__host__ __device__ constexpr bool has_class(int Q, int c2) {
    return c2 == 0 || c2 == 1 || (c2 == 2 && (Q == 19 || Q == 27)) || (c2 == 3 && (Q == 15 || Q == 27));
}

// compact index k of stencil Q -> D3Q27 index
__host__ __device__ constexpr int q_of(int Q, int k) {
    int n = 0;
    for (int q = 0; q < 27; ++q)
        if (has_class(Q, cls27(q))) {
            if (n == k) return q;
            ++n;
        }
    return -1;
}

// weight of class c2 in stencil Q (eqs. B.1-B.4)
__host__ __device__ constexpr double weight(int Q, int c2) {
    return Q == 27 ? (c2 == 0 ? 64.0 / 216 : c2 == 1 ? 16.0 / 216 : c2 == 2 ? 4.0 / 216 : 1.0 / 216)
         : Q == 19 ? (c2 == 0 ? 12.0 / 36 : c2 == 1 ? 2.0 / 36 : 1.0 / 36)
         : Q == 15 ? (c2 == 0 ? 16.0 / 72 : c2 == 1 ? 8.0 / 72 : 1.0 / 72)
                   : (c2 == 0 ? 0.0 : 1.0 / 6);
}

template <int I> struct IC { static constexpr int value = I; };
// compile-time loop: f(IC<I>{}) for I in [I0, N)
template <int I, int N, typename F>
__device__ __forceinline__ void static_for(F&& f) {
    if constexpr (I < N) {
        f(IC<I>{});
        static_for<I + 1, N>(static_cast<F&&>(f));
    }
}

}  // namespace tcp
