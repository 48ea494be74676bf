"""DRAM traffic per launch (dram__bytes_read.sum + dram__bytes_write.sum) of the hot kernels, copied
from the committed `ncu --set full` summaries under profiles/ (bench.py's `roofline.traffic` field: it
cannot be measured inside a timed run).  Keyed by BASELINE.json config index and bench leg."""

# profiles/r1_v4.md: fwd_cl_kernel<float> 121.4 + 32.4 MB; bwd_pull_kernel<float,true> 52.2 + 126.9 MB
# (+ pull_prep_kernel 0.06 MB).  Writes below the algorithmic bytes = output still dirty in L2 at kernel end.
TRAFFIC_BYTES = {
    2: {"fwd": 153_774_080, "bwd": 179_159_552, "source": "profiles/r1_v4.md"},
}
