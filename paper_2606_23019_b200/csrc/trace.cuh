// trace.cuh -- cycle-counter instrumentation of the forward kernel's roles, compiled in only with
// -DSA_TRACE (a debug build: the product kernel contains none of it). Each role keeps a set of
// accumulators; XX_TR(i) adds the clocks since the role's previous trace point to accumulator i, and
// the role prints per-unit / per-item averages for CTAs 0 and 1 when it ends. This is where the
// phase times quoted in DESIGN.md ("Measured on the way") come from.
#pragma once

#ifdef SA_TRACE
// ---- MMA issuer: 0 other, 1 wait for P, 2 wait for K, 3 wait for V / o_free, 4 scheduler / Q,
//      5 S issue, 6 PV issue
#define IT_TRACE_DECL uint32_t itr[7] = {0, 0, 0, 0, 0, 0, 0}, itl = clock(), it_units = 0;
#define IT_TR(i) { const uint32_t n_ = clock(); itr[i] += n_ - itl; itl = n_; }
#define IT_TRACE_UNIT ++it_units;
#define IT_TRACE_REPORT                                                                                  \
  if (lane == 0 && blockIdx.x < 2)                                                                       \
    printf("issuer cta %d units %u: other %u | p_full %u | K %u | V/o_free %u | sched/q %u | S issue %u " \
           "| PV issue %u (clk per unit)\n", blockIdx.x, it_units, itr[0] / it_units, itr[1] / it_units, \
           itr[2] / it_units, itr[3] / it_units, itr[4] / it_units, itr[5] / it_units, itr[6] / it_units);
// ---- softmax warpgroup: per block 0 other, 1 wait for S, 2 TMEM load, 3 row max + rescale,
//      4 exponentials + P store; per item 5 scheduler, 6 wait for Q, 7 row norms, 8 wait for the
//      last PV, 9 epilogue
#define SA_TRACE_DECL \
  uint32_t tr_acc[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0}, tr_last = clock(), tr_n = 0, tr_items = 0;
#define SA_TR(i) { const uint32_t now_ = clock(); tr_acc[i] += now_ - tr_last; tr_last = now_; if (i == 4) ++tr_n; }
#define SA_TRACE_ITEM ++tr_items;
#define SA_TRACE_REPORT                                                                                    \
  if (lane == 0 && blockIdx.x < 2 && quarter == 0)                                                         \
    printf("trace cta %d wg %d blocks %u: other %u | wait_s %u | ld %u | max+resc %u | exp+st %u (clk per " \
           "block); items %u: sched %u | q_full %u | norms %u | o_full %u | epilogue %u (clk per item)\n",  \
           blockIdx.x, t, tr_n, tr_acc[0] / tr_n, tr_acc[1] / tr_n, tr_acc[2] / tr_n, tr_acc[3] / tr_n,     \
           tr_acc[4] / tr_n, tr_items, tr_acc[5] / tr_items, tr_acc[6] / tr_items, tr_acc[7] / tr_items,    \
           tr_acc[8] / tr_items, tr_acc[9] / tr_items);
#else
#define IT_TRACE_DECL
#define IT_TR(i)
#define IT_TRACE_UNIT
#define IT_TRACE_REPORT
#define SA_TRACE_DECL
#define SA_TR(i)
#define SA_TRACE_ITEM
#define SA_TRACE_REPORT
#endif
