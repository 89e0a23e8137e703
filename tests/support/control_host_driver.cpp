// Host build of the device-side control flow (csrc/control.cuh) for the CPU tests: the same source,
// compiled by g++ with the CUDA qualifiers defined away.  Reads a scripted run from stdin and prints
// the decision taken before every layer.
//
//   line 1:  order nfields n_occ max_layers s1_autoscale
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
