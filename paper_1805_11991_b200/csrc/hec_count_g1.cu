// Count kernels of genus 1 (hec_count_kernels.cuh), one translation unit per genus so that they compile in parallel.
#define HEC_COUNT_GENUS 1
#include "hec_count_kernels.cuh"

int hec_launch_count_g1(LibState &S, const DevicePlan &plan, HecCountParams P) { return launch_count<1, 4>(S, plan, P); }
