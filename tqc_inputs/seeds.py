"""Seed convention (SURVEY.md section 8(d) "Seeds")."""

STREAM_LAYOUT = 0     # graph / network layout
STREAM_GATES = 1      # gate choices / angles
STREAM_TENSORS = 2    # tensor values
STREAM_STATES = 3     # bitstrings
STREAM_SUBSET = 4     # checked-subset indices


def seed_for(cfg: int, stream: int, bump: int = 0) -> int:
    """seed(cfg, stream) = 250203445*100 + 10*cfg + stream (+1000*bump for seed searches)."""
    return 250203445 * 100 + 10 * cfg + stream + 1000 * bump
