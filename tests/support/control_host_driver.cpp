// Host build of the device-side control flow (csrc/control.cuh) for the CPU tests: the same source,
// compiled by g++ with the CUDA qualifiers defined away.  Reads a scripted run from stdin and prints
// the decision taken before every layer.
//
//   line 1:  order nfields n_occ max_layers s1_autoscale      (order 11: the two sides of an order-parallel pair,
//                                                            each with its own DmptCtl, joined by the hand-off records)
//   line 2:  n_s n_x                      (Tr S0_0, ||S0_0||_F^2: what the transform kernel reports)
//   then one line per executed layer:  RED_COUNT doubles (the reductions the layer's epilogues wrote)
//
// Output, one line per decision:  layer sigma mode0 conv0 conv1 conv2 conv3 done status
#define __device__
#define __forceinline__ inline
#include <math.h>
#include <stdio.h>
#include <string.h>

#include "control.cuh"

using namespace dmpt;

int main() {
    DmptProblem pb;
    memset(&pb, 0, sizeof pb);
    DmptCtl c;
    memset(&c, 0, sizeof c);
    if (scanf("%d %d %d %d %d", &pb.order, &pb.nfields, &pb.n_occ, &pb.max_layers, &pb.s1_autoscale) != 5) return 2;
    if (scanf("%lf %lf", &c.n_s, &c.n_x) != 2) return 2;
    static int sigma[2048];
    static double tr_s[2048], tr_x[2048], id_err[2048], fro1[2048], fro2[2048], fro3[2048];
    DmptLogs L = {sigma, tr_s, tr_x, id_err, fro1, fro2, fro3};
    if (pb.order == 11) {
        // order-parallel pair: side A (order 0, pair_side 1) decides and publishes, side B (order 1, pair_side 2)
        // merges the record of its layer at the start of the launch and again in its control step - as the kernel does
        static int sigma_b[2048];
        static double trs_b[2048], trx_b[2048], ide_b[2048], fro1_b[2048], fro2_b[2048], fro3_b[2048];
        static DmptHandoff hand[2050];
        memset(hand, 0, sizeof hand);
        DmptLogs LB = {sigma_b, trs_b, trx_b, ide_b, fro1_b, fro2_b, fro3_b};
        DmptProblem pa = pb, pbb = pb;
        pa.order = 0; pa.pair_side = 1;
        pbb.order = 1; pbb.pair_side = 2;
        DmptCtl a = c, b;
        memset(&b, 0, sizeof b);
        a.layer = 1;
        control_decide(a, L, pa);
        handoff_publish(a, hand);
        b.layer = 1;
        for (;;) {
            DmptCtl seen = b;                       // what side B's launch of layer b.layer runs with
            handoff_merge(seen, hand[seen.layer]);
            printf("%d %d %d %d %d %d %d %d %d\n", seen.layer, seen.sigma, seen.mode0, seen.conv0, seen.conv1, 0, 0,
                   seen.done || b.done, seen.done ? seen.status : b.status);
            if (seen.done || b.done) break;
            double red[RED_COUNT];
            for (int k = 0; k < RED_COUNT; ++k)
                if (scanf("%lf", &red[k]) != 1) return 0;
            if (!a.done) control_finalize(a, L, pa, red, hand);          // side A runs one layer ahead at most
            handoff_merge(b, hand[b.layer]);
            control_finalize(b, LB, pbb, red, hand);
            if (b.done) {
                printf("%d %d %d %d %d %d %d %d %d\n", b.layer, b.sigma, b.mode0, b.conv0, b.conv1, 0, 0, 1, b.status);
                break;
            }
        }
        printf("end %d %d %d %d %d %.17g\n", b.layers, a.n_c, b.n_c1, 0, 0, a.fro0);
        return 0;
    }
    c.layer = 1;
    control_decide(c, L, pb);                      // what dmpt_control_init_kernel does
    for (;;) {
        printf("%d %d %d %d %d %d %d %d %d\n", c.layer, c.sigma, c.mode0, c.conv0, c.conv1, c.conv2, c.conv3, c.done,
               c.status);
        if (c.done) break;
        double red[RED_COUNT];
        for (int k = 0; k < RED_COUNT; ++k)
            if (scanf("%lf", &red[k]) != 1) return 0;    // script exhausted
        control_finalize(c, L, pb, red);
    }
    printf("end %d %d %d %d %d %.17g\n", c.layers, c.n_c, c.n_c1, c.n_c2, c.n_c3, c.fro0);
    return 0;
}
