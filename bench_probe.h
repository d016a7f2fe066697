/*
 * bench_probe.h -- the one call of libzmc_probe.so, bench.py's micro-benchmark of the SM's dispatch costs (bench_probe.cu).
 * Not part of the zmc_scan library: nothing in include/zmc.h or libzmc.so refers to it.
 */
#ifndef BENCH_PROBE_H_
#define BENCH_PROBE_H_
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

/* One measured row.  All three numbers are SM-sub-partition cycles per group of instructions per warp. */
#define BENCH_PIPE_MAX_ROWS 48
typedef struct bench_pipe_row {
    char name[72];           /* e.g. "LOP3", "1xIMAD.WIDE+LOP3 + 2xDFMA, same warp", "cfg2 block: both, same warp (ptxas order)" */
    double cycles;           /* measured */
    double parallel;         /* max of the parts' own costs: what independent pipes would give */
    double serial;           /* sum of the parts' own costs: what one shared pipe would give */
} bench_pipe_row;
typedef struct bench_pipe_report {
    double sm_mhz;           /* SM clock while measuring (clock64 against globaltimer) */
    int32_t sm_count;
    int32_t n_rows;
    bench_pipe_row rows[BENCH_PIPE_MAX_ROWS];
} bench_pipe_report;

/* Runs ~35 short synthetic kernels (about 0.1 s) on `stream` (a cudaStream_t) of the current device and synchronises: the
 * dispatch cost of every instruction class the hot loop uses, which pairs of classes overlap (in one warp, and across
 * warps), and cfg 2's instruction mix per Philox block.  Returns 0, a cudaError_t, or -1 for a NULL report. */
int bench_measure_pipes(bench_pipe_report* report, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* BENCH_PROBE_H_ */
