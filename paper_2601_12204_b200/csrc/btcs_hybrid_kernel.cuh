// btcs_hybrid_kernel.cuh -- the body of the HYBRID kernel for N == P * threads; included TWICE by btcs_hybrid.cu
// (no include guard) with BURGERS_HYBRID_NAME / BURGERS_HYBRID_BOUNDS set to the entry point's name and its
// __launch_bounds__: the same code is needed with and without a register cap, and neither a second launch-bound
// argument that depends on a template parameter nor a __forceinline__ body shared by two __global__ wrappers
// leaves the instruction schedule of the 128-thread instances alone (see btcs_hybrid.cu).
// TN: the thread count as a compile-time constant (0: blockDim.x).  With TN known the PCR levels are unrolled and
// every shared-memory index is an immediate offset from two registers; the run-time form spends 50 of the 64
// instructions of a level on address arithmetic, and the kernel is bound by issue slots (an FP64 instruction
// takes two): C3 15.66 -> 14.2 ms.
// DIRI: Dirichlet ends (identity rows 0 and N - 1); the periodic instances carry no row selects.
template <typename T, int P, int TN, bool DIRI>
__global__ void BURGERS_HYBRID_BOUNDS
BURGERS_HYBRID_NAME(T *__restrict__ u, const T *__restrict__ nu, const T *__restrict__ dt, int N,
                   double inv_dx, int64_t n_steps, int bc) {
    constexpr int V = 16 / sizeof(T);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int t = threadIdx.x, Tn = TN ? TN : (int)blockDim.x, mask = Tn - 1;
    T *sA = reinterpret_cast<T *>(smem_raw);  // [2][Tn] reduced rows (PCR ping-pong)
    T *sC = sA + 2 * Tn;
    T *sD = sC + 2 * Tn;
    T *sFA = sD + 2 * Tn;                     // [Tn] first interface rows (cyclic-reduction step)
    T *sFC = sFA + Tn;
    T *sFD = sFC + Tn;
    T *row = u + (int64_t)blockIdx.x * N + (int64_t)t * P;

    Coef<T> co;
    co.init(nu[blockIdx.x], dt[blockIdx.x], inv_dx);
    (void)bc;
    const bool fixL = DIRI && t == 0;
    const bool fixR = DIRI && t == Tn - 1;

    T v[P];
#pragma unroll
    for (int c = 0; c < P / V; ++c) {
        int4 q4 = *reinterpret_cast<const int4 *>(row + c * V);
        const T *e = reinterpret_cast<const T *>(&q4);
#pragma unroll
        for (int k = 0; k < V; ++k) v[c * V + k] = e[k];
    }

    for (int64_t n = 0; n < n_steps; ++n) {
        T f[P], c[P], q[P];
        // ---- assembly + partition elimination
        Row<T> first, last;
        eliminate<T, P>(v, co, [&](int j) { return (j == 0 && fixL) || (j == P - 1 && fixR); },
                        f, c, q, first, last);
        // ---- cyclic-reduction step: substitute the x_0 rows of threads t and t+1 into the x_L row
        // of thread t:  [-f A] x_L(t-1) + [1 - f C - c A'] x_L(t) + [-c C'] x_L(t+1) = q - f D - c D'
        sFA[t] = first.A; sFC[t] = first.C; sFD[t] = first.D;
        __syncthreads();
        Row<T> r;
        {
            const int tn = (t + 1) & mask;
            const T nA = sFA[tn], nC = sFC[tn], nD = sFD[tn];
            const T m = rcp(t_fma(-last.A, first.C, t_fma(-last.C, nA, T(1))));
            r.A = -last.A * first.A * m;
            r.C = -last.C * nC * m;
            r.D = t_fma(-last.A, first.D, t_fma(-last.C, nD, last.D)) * m;
        }
        int cur = 0;
        sA[t] = r.A; sC[t] = r.C; sD[t] = r.D;
        __syncthreads();
        // ---- parallel cyclic reduction over the Tn reduced rows (cyclic chain), early exit
        bool finished = false;
#pragma unroll
        for (int s = 1; s < Tn / 2; s <<= 1) {
            const int km = (t - s) & mask, kp = (t + s) & mask;
            const T *pA = sA + cur * Tn, *pC = sC + cur * Tn, *pD = sD + cur * Tn;
            Row<T> rm, rp;
            rm.A = pA[km]; rm.C = pC[km]; rm.D = pD[km];
            rp.A = pA[kp]; rp.C = pC[kp]; rp.D = pD[kp];
            r = pcr_combine(r, rm, rp);
            const int o = (cur ^ 1) * Tn + t;
            sA[o] = r.A; sC[o] = r.C; sD[o] = r.D;
            cur ^= 1;
            // The vote starts at the third level: no set of coefficients worth a fast path is done before, and a
            // vote costs the read-back of the barrier's result and a dependent branch (C3: 13.88 -> 13.45 ms);
            // levels past the decoupling change the right-hand sides by less than 2^-70 of their neighbours'.
            if (s >= 4) {
                const int flag = !((t_abs(r.A) <= Lim<T>::tiny()) & (t_abs(r.C) <= Lim<T>::tiny()));
                if (!__syncthreads_or(flag)) { finished = true; break; }
            } else {
                __syncthreads();
            }
        }
        T xL = r.D, xLprev;
        if (finished) {
            xLprev = sD[cur * Tn + ((t - 1) & mask)];
        } else {  // rows t and t + Tn/2 couple only to each other: exact 2x2 solve
            const int o = (t + Tn / 2) & mask;
            const T p1 = r.A + r.C, p2 = sA[cur * Tn + o] + sC[cur * Tn + o];
            const T D2 = sD[cur * Tn + o];
            xL = t_fma(-p1, D2, r.D) * rcp(t_fma(-p1, p2, T(1)));
            sD[(cur ^ 1) * Tn + t] = xL;   // the other PCR buffer is free; its next write follows a barrier
            __syncthreads();
            xLprev = sD[(cur ^ 1) * Tn + ((t - 1) & mask)];
        }
        // ---- recover x_0 and back-substitute
        const T x0 = t_fma(-first.A, xLprev, t_fma(-first.C, xL, first.D));
        back_substitute<T, P>(v, f, c, q, x0, xL);
    }

#pragma unroll
    for (int c = 0; c < P / V; ++c) {
        int4 q4;
        T *e = reinterpret_cast<T *>(&q4);
#pragma unroll
        for (int k = 0; k < V; ++k) e[k] = v[c * V + k];
        *reinterpret_cast<int4 *>(row + c * V) = q4;
    }
}

