// Lattice velocity sets as compile-time tables (Tables 1-3; D3Q7: DESIGN.md R6).
// Every kernel unrolls over directions with the index as a template constant, so c_i, the
// weight class and the opposite direction fold into immediate operands.
#pragma once
#include <type_traits>

namespace lbm {

// compile-time loop: f(std::integral_constant<int, I>) for I in [B, E)
template <int B, int E, class F>
__host__ __device__ __forceinline__ void static_for(F&& f) {
    if constexpr (B < E) {
        f(std::integral_constant<int, B>{});
        static_for<B + 1, E>(f);
    }
}

// D3Q19, Table 1 as printed: rest, 6 axis, 12 face diagonals; opposite pairs (2k-1, 2k)
struct D3Q19 {
    static constexpr int Q = 19, D = 3;
    __host__ __device__ static constexpr int c(int i, int a) {
        constexpr int t[19][3] = {{0, 0, 0},   {1, 0, 0},  {-1, 0, 0},  {0, 1, 0},  {0, -1, 0}, {0, 0, 1},  {0, 0, -1},
                                  {1, 1, 0},   {-1, -1, 0}, {1, 0, 1},  {-1, 0, -1}, {0, 1, 1},  {0, -1, -1},
                                  {1, -1, 0},  {-1, 1, 0},  {1, 0, -1}, {-1, 0, 1},  {0, 1, -1}, {0, -1, 1}};
        return t[i][a];
    }
    __host__ __device__ static constexpr int opp(int i) { return i == 0 ? 0 : ((i & 1) ? i + 1 : i - 1); }
    // weight class: 0 rest (1/3), 1 axis (1/18), 2 diagonal (1/36)
    __host__ __device__ static constexpr int wclass(int i) { return i == 0 ? 0 : (i <= 6 ? 1 : 2); }
    __host__ __device__ static constexpr double w(int i) { return i == 0 ? 1.0 / 3.0 : (i <= 6 ? 1.0 / 18.0 : 1.0 / 36.0); }
};

// D2Q9, Table 2; w_4 = 1/9 (the printed 1/36 breaks sum w = 1; R1)
struct D2Q9 {
    static constexpr int Q = 9, D = 2;
    __host__ __device__ static constexpr int c(int i, int a) {
        constexpr int t[9][3] = {{0, 0, 0}, {1, 0, 0}, {0, 1, 0}, {-1, 0, 0}, {0, -1, 0},
                                 {1, 1, 0}, {-1, 1, 0}, {-1, -1, 0}, {1, -1, 0}};
        return t[i][a];
    }
    __host__ __device__ static constexpr int opp(int i) { return i == 0 ? 0 : (i <= 4 ? ((i + 1) % 4) + 1 : ((i - 3) % 4) + 5); }
    __host__ __device__ static constexpr int wclass(int i) { return i == 0 ? 0 : (i <= 4 ? 1 : 2); }
    __host__ __device__ static constexpr double w(int i) { return i == 0 ? 4.0 / 9.0 : (i <= 4 ? 1.0 / 9.0 : 1.0 / 36.0); }
};

// scalar lattices: D2Q5, Table 3; D3Q7 in the order of D3Q19's first seven (R6).
// Weights are runtime (w0_scalar is a parameter): w_0 = w0, w_{i>0} = (1-w0)/(Q-1).
struct D2Q5 {
    static constexpr int Q = 5, D = 2;
    __host__ __device__ static constexpr int c(int i, int a) {
        constexpr int t[5][3] = {{0, 0, 0}, {1, 0, 0}, {0, 1, 0}, {-1, 0, 0}, {0, -1, 0}};
        return t[i][a];
    }
    __host__ __device__ static constexpr int opp(int i) { return i == 0 ? 0 : ((i + 1) % 4) + 1; }
};
struct D3Q7 {
    static constexpr int Q = 7, D = 3;
    __host__ __device__ static constexpr int c(int i, int a) {
        constexpr int t[7][3] = {{0, 0, 0}, {1, 0, 0}, {-1, 0, 0}, {0, 1, 0}, {0, -1, 0}, {0, 0, 1}, {0, 0, -1}};
        return t[i][a];
    }
    __host__ __device__ static constexpr int opp(int i) { return i == 0 ? 0 : ((i & 1) ? i + 1 : i - 1); }
};

template <class L> struct ScalarOf;
template <> struct ScalarOf<D2Q9> { using type = D2Q5; };
template <> struct ScalarOf<D3Q19> { using type = D3Q7; };

}  // namespace lbm
