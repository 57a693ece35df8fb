"""CPU oracle for the Exa.TrkX inference hot path -- TEST INFRASTRUCTURE, NOT PRODUCT.

A plain, slow, fp64 NumPy restatement of the five stages of PAPER.md line 85 (section
2.2.2): embedding MLP -> fixed-radius graph in the latent space -> filter MLP +
threshold -> interaction-network GNN edge scores -> weakly-connected components.  The
paper gives the stage order only; every number (widths, radius, caps, cuts, equations
of the interaction network) follows BASELINE.json `configs` and the readings C-1..C-22
of SURVEY.md section 8(c), restated in DESIGN.md.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package.  It shares no code with paper_2501_05520_b200/ (the CUDA path)
and neither imports the other; both read inputs from synth/.

Library primitives used as steps: numpy matmul (fp64 BLAS), argsort/lexsort, add.at.
There is no blocking, fusion or reordering beyond what the definitions state; the
query/cell chunking in s2_frnn only bounds memory and does not change any result.

Pins (tests/test_oracle_*.py, -m "not gpu"): see DESIGN.md section "Oracle pins".
parity unpinned: the end-to-end physics quality of the whole pipeline (trained weights
and the paper's events are not available).  Every stage function
is pinned on its own.
"""
from . import s1_embed, s2_frnn, s3_filter, s4_gnn, s5_cc, s6_tracks  # noqa: F401
from .mlp import layernorm, linear, mlp_forward, sigmoid  # noqa: F401
