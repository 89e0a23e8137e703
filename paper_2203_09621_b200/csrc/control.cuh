// Device-resident scalar state and control flow of Algorithms 1-3.
//
// The per-layer decisions (sigma_n, the D0 test of Algorithm 2, the D1/D2 tests of Algorithm 3,
// loop exit) are taken on the device by the LAST CTA of each layer launch ("finalizer"), from
// fp64 sums of the fp32 per-CTA partial reductions the epilogues wrote.  The next launch reads
// the decision from DmptCtl at kernel start; the host never sees a scalar until the run ends.
//
// Reading R9: N_X = Tr[(S0_{n-1})^2] is evaluated as ||S0_{n-1}||_F^2 (equal for a
// symmetric matrix) and N_S as the actual trace of the stored S0_{n-1}; both are accumulated by
// the epilogue that WRITES S0_{n-1}, so sigma_n and the D0 decision of layer n are known before
// layer n's products start.
#pragma once
#include <math.h>
#include <stdint.h>

namespace dmpt {

constexpr double kCD0 = 4.5;   // PAPER.md:518 (Algorithm 2)
constexpr double kCPT = 9.0;   // PAPER.md:465, 524 (Algorithm 3)

// slots of the per-warp partial reductions written by the layer epilogue
enum Red : int {
    RED_TR_S0 = 0,   // sum of the new S0 diagonal                      -> N_S
    RED_FRO_S0 = 1,  // sum of squares of the new S0                    -> N_X of the next layer
    RED_FRO0 = 2,    // sum (S0 - X0)^2 on the D0 stop layer            -> FroErr0^2
    RED_FRO1 = 3,    // sum (S1 - X1)^2 once D0 converged               -> FroErr1_n^2
    RED_MAX1 = 4,    // max |new S1|                                    -> next S1 scale
    RED_FRO2 = 5,    // sum (S2 - X2)^2 once D1 converged (order 2)     -> FroErr2_n^2
    RED_MAX2 = 6,    // max |new S2|
    RED_FRO3 = 7,    // third response slot (multi-field runs only)
    RED_MAX3 = 8,
    RED_COUNT = 10
};
// Response slots.  Slot 1 is S1 of the (first) perturbation.  Slot 2 is S2 at order 2, or S1 of a SECOND
// perturbation sharing H0 in a multi-field first-order run (the x, y, z fields of the
// polarizability, Eq. 79); slot 3 is S1 of a third perturbation.

enum Mode0 : int { MODE_ACTIVE = 0, MODE_STOP = 1, MODE_FROZEN = 2 };

struct DmptCtl {
    // ---- decision for the next layer launch
    int layer;      // n of the layer the next launch executes (1-based)
    int done;       // launches exit at once when set
    int status;     // DMPT_OK or a negative DMPT_E* code
    int mode0;      // Mode0
    int sigma;      // sigma_n
    int s0_buf;     // hi/lo buffer holding S0_{n-1}
    int s1_buf;     // fp32 + hi/lo buffer holding S1_{n-1}
    int s2_buf;
    int s3_buf;
    int e1_in;      // S1 operand buffers hold fp16(2^e1_in S1_{n-1})
    int e1_out;     // scale for the split of S1_n
    int e2_in, e2_out;
    int e3_in, e3_out;
    int p1, p2, p3; // prescale exponents: slot k holds 2^pk times the true response iterate (0 unless |H1|/W is
                    // outside [2^-30, 2^30]; at order 2 slot 2 then holds 2^(2 p1) S2)
    // ---- state of Algorithms 1-3
    int conv0, conv1, conv2, conv3;
    int n_c, n_c1, n_c2, n_c3;
    int layers;     // layers executed so far
    int single_shot;  // 1: dmpt_layer_products - run one layer, take no decisions
    unsigned int ticket;  // CTA arrival counter of the running launch
    unsigned int wave;    // wave-boundary arrivals of the running launch (LayerParams::wave_sync)
    unsigned int wave2;   // the same for the order-2 pass of the layer
    unsigned int wave3;   // the same for the order-3 pass of the layer
    double n_s;     // Tr S0_{n-1}
    double n_x;     // ||S0_{n-1}||_F^2
    double fro0;    // FroErr0
    double eps_min, eps_max;
    double s1_max, s2_max, s3_max;
};

struct DmptLogs {   // device arrays, max_layers entries, entry n-1 for layer n
    int* sigma;
    double* tr_s;
    double* tr_x;
    double* id_err;
    double* fro1;
    double* fro2;
    double* fro3;
    struct DmptClockStamps* clk;     // SM clock stamps of the layer launches (may be null)
};

// (clock64, globaltimer) of every SM at the start of the first and of the latest order-0 launch of a run: their
// difference is the SM clock the layer loop really ran at (dmpt_result.sm_clock_mhz).  Under the power cap it is
// well below what nvidia-smi samples show.
constexpr int kMaxSmStamps = 256;
struct DmptClockStamps {
    long long first[kMaxSmStamps][2];
    long long last[kMaxSmStamps][2];
};

struct DmptProblem {
    int n, n_pad, n_occ, order, max_layers, s0_shift, s1_autoscale;
    int nfields;     // 1..3 perturbations sharing H0 (order 1 only above 1)
    int pair_side;   // order-parallel pair: 0 = the whole path on one device;
                     // 1 = the order-0 side (S0^2, sigma_n, Algorithm 2); 2 = the order-1 side (S0.S1 + S1.S0, Algorithm 3)
};

// Order-parallel pair: what the order-0 side hands to the order-1 side for layer n, next to the operand pair
// (Mhi, Mlo) of S0_{n-1}.  One record per layer, written by the order-0 side's control step when it decides layer n,
// copied device to device, read by the order-1 side's launch of layer n.  valid = 0: the order-0 side had already
// finished (S0 frozen) - the order-1 side then flips sigma itself.
struct DmptHandoff {
    int valid;
    int sigma;      // sigma_n
    int conv0;      // Algorithm 2 has fired (on layer n or before): FroErr1_n is wanted
    int n_c;
    int s0_buf;     // operand buffer holding M of S0_{n-1}
    int done;       // the order-0 side stopped with an error (status below)
    int status;
    int pad_;
    double fro0;    // FroErr0 (known from layer n_c + 1 on)
};

// exact power of two 2^e bringing m into [8, 16); 0 when m is 0 or not finite
__device__ __forceinline__ int scale_exponent(double m) {
    if (!(m > 0.0) || !isfinite(m)) return 0;
    int e;
    frexp(m, &e);          // m = f * 2^e, f in [0.5, 1)  ->  m in [2^(e-1), 2^e)
    e = 4 - e;             // m * 2^(4-e) in [8, 16)
    // every factor 2^(+-e), 2^(+-2e) of the layer epilogue must stay a normal fp32 number; the prescale of
    // dmpt_bounds_to_ctl_kernel keeps |e| far inside this range on every input
    return e < -48 ? -48 : (e > 48 ? 48 : e);
}

// Decide layer n = ctl.layer from N_S, N_X (PAPER.md:499-505 and Algorithm 2).
__device__ inline void control_decide(DmptCtl& c, const DmptLogs& L, const DmptProblem& pb) {
    const int n = c.layer;
    if (n > pb.max_layers) {
        c.done = 1;
        c.status = -5;  // DMPT_ENOCONV
        return;
    }
    L.tr_s[n - 1] = c.n_s;
    if (!c.conv0) {
        const double n_s = c.n_s, n_x = c.n_x, nocc = (double)pb.n_occ;
        const double ide = n_s - n_x;
        const int s = (fabs(2.0 * n_s - n_x - nocc) >= fabs(n_x - nocc)) ? 1 : -1;  // R3: tie -> +1
        L.tr_x[n - 1] = n_x;
        L.id_err[n - 1] = ide;
        L.sigma[n - 1] = s;
        if (!isfinite(n_s) || !isfinite(n_x)) {
            c.done = 1;
            c.status = -6;  // DMPT_ENUMERIC
            return;
        }
        bool stop = !(ide > 0.0);                                              // R6
        if (!stop && n > 2 && L.sigma[n - 2] != L.sigma[n - 3]) {
            const double prev = L.id_err[n - 3];
            stop = !(ide <= kCD0 * prev * prev);
        }
        c.sigma = s;
        if (stop) {
            c.conv0 = 1;
            c.n_c = n;
            c.mode0 = MODE_STOP;      // X0 is still formed once, for FroErr0 (R4)
            if (pb.order == 0 && pb.pair_side == 0) {      // ground-state mode: D0 = S0_{n-1} is the answer, nothing left to measure
                c.layers = n;         // counted like the oracle's loop: the pass on which the test fired
                c.fro0 = nan("");
                c.done = 1;
            }
        } else {
            c.mode0 = MODE_ACTIVE;
        }
    } else {
        const int s = -L.sigma[n - 2];
        L.sigma[n - 1] = s;
        L.tr_x[n - 1] = nan("");
        L.id_err[n - 1] = nan("");
        c.sigma = s;
        c.mode0 = MODE_FROZEN;
    }
}

// One response slot after layer n: record FroErr_n = ||S - X||_F once its gate opened (D0 converged for a
// first-order slot, D1 converged for the second-order slot), run the test of Algorithm 3 from
// `gate_layer + 2` on (R5, R6), and accept the new iterate unless the test fired.
__device__ inline void response_step(DmptCtl& c, const DmptProblem& pb, int n, bool gate, int gate_layer, int& conv,
                                     int& n_conv, int& buf, int& e_in, int& e_out, double& mx, double fro_sq,
                                     double max_new, double* log) {
    const double nanv = nan("");
    if (conv) {
        log[n - 1] = nanv;
        return;
    }
    if (gate) {
        const double f = sqrt(fro_sq);
        log[n - 1] = f;
        if (n - 2 >= gate_layer && !(f < kCPT * c.fro0 * log[n - 3])) {
            conv = 1;
            n_conv = n;
        }
        if (!isfinite(f) || !isfinite(c.fro0)) c.status = -6;
    } else {
        log[n - 1] = nanv;
    }
    if (!conv) {   // accept the new iterate
        buf ^= 1;
        e_in = e_out;
        mx = max_new;
        if (pb.s1_autoscale) e_out = scale_exponent(mx);
        if (!isfinite(mx)) c.status = -6;
    }
}

// Order-parallel pair, order-1 side: overlay the order-0 side's decision for layer c.layer on the local state.
// This side never forms S0^2: for its launch S0 is always "frozen", whatever the other side is doing with it.
__device__ inline void handoff_merge(DmptCtl& c, const DmptHandoff& h) {
    c.mode0 = MODE_FROZEN;
    if (!h.valid) return;
    c.sigma = h.sigma;
    c.conv0 = h.conv0;
    c.n_c = h.n_c;
    c.s0_buf = h.s0_buf;
    c.fro0 = h.fro0;
    if (h.done && h.status != 0) {
        c.done = 1;
        c.status = h.status;
    }
}

// Order-0 side: publish the decision just taken for layer c.layer.
__device__ inline void handoff_publish(const DmptCtl& c, DmptHandoff* out) {
    DmptHandoff h;
    h.valid = 1;
    h.sigma = c.sigma;
    h.conv0 = c.conv0;
    h.n_c = c.n_c;
    h.s0_buf = c.s0_buf;
    h.done = c.done;
    h.status = c.status;
    h.pad_ = 0;
    h.fro0 = c.fro0;
    out[c.layer] = h;
}

// After layer n = ctl.layer ran: fold its reductions into the state, apply Algorithm 3
// (cascade for orders 2 and 3, reading R15) and decide layer n+1.
// `handoff`: order-parallel pair only (DmptProblem::pair_side): the records the order-0 side writes (side 1) or the
// copies of them the order-1 side reads (side 2; the caller has already merged handoff[n] into c).
__device__ inline void control_finalize(DmptCtl& c, const DmptLogs& L, const DmptProblem& pb,
                                        const double* red /* RED_COUNT sums */, DmptHandoff* handoff = nullptr) {
    const int n = c.layer;
    c.layers = n;
    if (c.single_shot) {
        c.done = 1;
        return;
    }
    if (c.mode0 == MODE_ACTIVE) {
        c.n_s = red[RED_TR_S0];
        c.n_x = red[RED_FRO_S0];
        c.s0_buf ^= 1;
    } else if (c.mode0 == MODE_STOP) {
        c.fro0 = sqrt(red[RED_FRO0]);
    }
    if (pb.pair_side == 1) {
        // ---- order-0 side of a pair: after the stop layer (FroErr0 measured) nothing is left to do here; the
        //      last record tells the other side that S0 is frozen and what FroErr0 is
        L.fro1[n - 1] = nan("");
        if (c.mode0 == MODE_STOP) {
            if (!isfinite(c.fro0)) c.status = -6;
            c.layer = n + 1;
            c.sigma = -c.sigma;
            c.mode0 = MODE_FROZEN;
            c.done = 1;
            handoff_publish(c, handoff);
            return;
        }
        c.layer = n + 1;
        control_decide(c, L, pb);
        handoff_publish(c, handoff);
        return;
    }
    if (pb.pair_side == 2) L.sigma[n - 1] = c.sigma;       // this side's log: the flips after the freeze start from it
    // ---- first order (slot 1): Algorithm 3, tested from layer n_c + 2 on
    if (pb.order >= 1)
        response_step(c, pb, n, c.conv0 != 0, c.n_c, c.conv1, c.n_c1, c.s1_buf, c.e1_in, c.e1_out, c.s1_max,
                      red[RED_FRO1], red[RED_MAX1], L.fro1);
    else
        L.fro1[n - 1] = nan("");
    if (pb.order >= 2) {
        // ---- second order (slot 2): the same test cascaded behind the D1 stop (reading R15)
        response_step(c, pb, n, c.conv1 != 0, c.n_c1, c.conv2, c.n_c2, c.s2_buf, c.e2_in, c.e2_out, c.s2_max,
                      red[RED_FRO2], red[RED_MAX2], L.fro2);
        // ---- third order (slot 3): cascaded once more, behind the D2 stop
        if (pb.order >= 3)
            response_step(c, pb, n, c.conv2 != 0, c.n_c2, c.conv3, c.n_c3, c.s3_buf, c.e3_in, c.e3_out, c.s3_max,
                          red[RED_FRO3], red[RED_MAX3], L.fro3);
    } else if (pb.nfields >= 2) {
        // ---- further first-order fields (slots 2, 3): each runs Algorithm 3 on its own, like slot 1
        response_step(c, pb, n, c.conv0 != 0, c.n_c, c.conv2, c.n_c2, c.s2_buf, c.e2_in, c.e2_out, c.s2_max,
                      red[RED_FRO2], red[RED_MAX2], L.fro2);
        if (pb.nfields >= 3)
            response_step(c, pb, n, c.conv0 != 0, c.n_c, c.conv3, c.n_c3, c.s3_buf, c.e3_in, c.e3_out, c.s3_max,
                          red[RED_FRO3], red[RED_MAX3], L.fro3);
    }
    if (c.status != 0) {
        c.done = 1;
        return;
    }
    const bool all_fields = c.conv1 && (pb.nfields < 2 || c.conv2) && (pb.nfields < 3 || c.conv3);
    if (pb.order == 3 ? c.conv3 != 0 : (pb.order == 2 ? c.conv2 != 0 : (pb.order == 1 && all_fields))) {
        c.done = 1;
        return;
    }
    c.layer = n + 1;
    if (pb.pair_side == 2 && !c.conv0) {
        // the decision for layer n + 1 arrives from the order-0 side with that layer's operands
        if (c.layer > pb.max_layers) {
            c.done = 1;
            c.status = -5;  // DMPT_ENOCONV
        }
        return;
    }
    control_decide(c, L, pb);
}

}  // namespace dmpt
