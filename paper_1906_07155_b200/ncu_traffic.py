"""DRAM traffic per launch (dram__bytes_read.sum + dram__bytes_write.sum) of the hot kernels, copied
from the committed `ncu --set full` summaries under profiles/ (bench.py's `roofline.traffic` field: it
cannot be measured inside a timed run).  Keyed by BASELINE.json config index and bench leg."""

# profiles/r1_v5.md: fwd_cl_kernel<float> (with the prep blocks) 121.9 + 34.1 MB; bwd_pull_kernel<float,true>
# 56.5 + 131.6 MB.  Writes below the algorithmic bytes = output still dirty in L2 at kernel end.
TRAFFIC_BYTES = {
    2: {"fwd": 155_990_016, "bwd": 188_186_368, "source": "profiles/r1_v5.md"},
}
