// Count kernels of genus 3 (hec_count_kernels.cuh), one translation unit per genus so that they compile in parallel.
#define HEC_COUNT_GENUS 3
#include "hec_count_kernels.cuh"

int hec_launch_count_g3(LibState &S, const DevicePlan &plan, HecCountParams P) { return launch_count<3, 4>(S, plan, P); }
