// Count kernels of genus 4 (hec_count_kernels.cuh), one translation unit per genus so that they compile in parallel.
#define HEC_COUNT_GENUS 4
#include "hec_count_kernels.cuh"

int hec_launch_count_g4(LibState &S, const DevicePlan &plan, HecCountParams P) { return launch_count<4, 4>(S, plan, P); }
