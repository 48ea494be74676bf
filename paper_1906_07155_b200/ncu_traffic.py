"""DRAM traffic per launch (dram__bytes_read.sum + dram__bytes_write.sum) of the hot kernels, copied
from the committed `ncu --set full` summaries under profiles/ (bench.py's `roofline.traffic` field: it
cannot be measured inside a timed run).  Keyed by BASELINE.json config index and bench leg."""

# profiles/r1_v6.md: fwd_cl_kernel<float,224> (with the prep blocks) 122.3 + 34.2 MB; bwd_pull_kernel<float,true>
# 56.5 + 129.9 MB.  Writes below the algorithmic bytes = output still dirty in L2 at kernel end.
TRAFFIC_BYTES = {
    2: {"fwd": 156_569_856, "bwd": 186_424_832, "source": "profiles/r1_v6.md"},
}
