// Count kernels of genus 2 (hec_count_kernels.cuh), one translation unit per genus so that they compile in parallel.
#define HEC_COUNT_GENUS 2
#include "hec_count_kernels.cuh"

int hec_launch_count_g2(LibState &S, const DevicePlan &plan, HecCountParams P) { return launch_count<2, 4>(S, plan, P); }
