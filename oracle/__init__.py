"""CPU oracle for the STARK decode path -- TEST INFRASTRUCTURE, NOT PRODUCT.

What it is: a plain, slow, obviously-correct fp64 implementation of
*conventional* semantic-ID beam search (§3.6 first two
paragraphs): beams are expanded along the batch dimension, every beam owns a
physically replicated copy of the prefix KV cache, attention is the ordinary
full-sequence softmax attention of one query over that beam's own cache, and
after each selection the caches are deep-copied into the new beam order.  STARK
"preserves the decoding results of standard beam search",
so this definition is what the CUDA path must reproduce.

A second, independent formulation (the paper's own: sequence-dimension
expansion under the tree mask of Eq. 14) lives in
`oracle/tree.py` and is checked against the first in `tests/`.

Rules (task statement, section 3):
  * only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` /
    `--impl reference` legs may import this package;
  * it shares no code with `paper_2607_04068_b200/`; neither imports the other;
    only `workloads/` (seeded input draws, no arithmetic) serves both;
  * no expected value here ever comes from the CUDA path.

Precision: fp64 everywhere except the beam-selection key, which is a single
fp32 addition `fl32(score + logp)` (SURVEY.md §8c O4 / DESIGN.md reading R4):
an fp64 key would break ties that fp32 creates and make bit-exact selection
parity impossible.

Pins (tests/test_oracle_*.py, `-m "not gpu"`): every function below is pinned
to something other than itself -- see DESIGN.md §5.  Nothing here is "parity
unpinned".
"""
from .attention import (  # noqa: F401
    softmax_attention_single,
    beam_attention,
    masked_attention,
)
from .selection import log_softmax_fp32, select_beams  # noqa: F401
from .beam_search import conventional_beam_search, BeamTrace  # noqa: F401
from .tree import ancestor_chains, tree_mask, sequence_expanded_attention  # noqa: F401
from .replay import replay_step_attention, replay_beam_attention  # noqa: F401
from .brute_force import enumerate_all_paths  # noqa: F401
from .encdec import (  # noqa: F401
    cross_attention, target_attention, self_tree_attention, cross_plus_self_attention, path_hidden_states,
)
