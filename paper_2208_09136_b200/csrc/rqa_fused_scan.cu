// rqa_fused_scan.cu — the diagonal scan of rqa_line.cu built a second time with the candidate log switched on
// (RQA_LINE_LOG): every line_scan_kernel instantiation here also appends the cells inside the sample brackets of the fused
// sweep (rqa_select.cu: run_sweep_fused) to a per-series list.  A separate translation unit so that the two sets of
// kernel instantiations compile side by side.
#define RQA_LINE_LOG 1
#include "rqa_line.cu"
