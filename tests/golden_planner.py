"""The three hand-worked planner networks and the loader of tests/golden/planner_steps.txt (shared by the oracle-side and
the library-side planner tests)."""
import os

from tqc_inputs.network import Network

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")

PLANNER_NETS = {
    "fig5": lambda: Network(4, [(0, 1), (1, 2), (1, 3), (2, 3)], [[0], [0, 1, 2], [1, 3], [2, 3]], [[0], [1], [2], [3]]),
    "five": lambda: Network(5, [(0, 1), (0, 1), (1, 2), (2, 3), (3, 4), (2, 4)],
                            [[0, 1], [0, 1, 2], [2, 3, 5], [3, 4], [4, 5]], [[0], [1], [2], [3], [4]]),
    "sigma_first": lambda: Network(4, [(0, 1)] * 4 + [(1, 3), (2, 3)],
                                   [[0, 1, 2, 3], [0, 1, 2, 3, 4], [5], [4, 5]], [[0], [1], [2], [3]]),
}


def golden_planner_steps():
    out = {}
    for line in open(os.path.join(GOLDEN, "planner_steps.txt")):
        if not line.strip() or line.startswith("#"):
            continue
        head, inner, ol, orr = [x.split() for x in line.split("|")]
        out.setdefault(head[0], []).append(dict(lhs=int(head[1]), rhs=int(head[2]), log2cost=int(head[3]),
                                                inner=[int(x) for x in inner], outer_lhs=[int(x) for x in ol],
                                                outer_rhs=[int(x) for x in orr]))
    return out
