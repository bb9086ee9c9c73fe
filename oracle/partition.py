"""The paper's tensor partitioning scheme (Alg. 1), plain Python.  TEST INFRASTRUCTURE ONLY.

The algorithm's body is missing from PAPER.md (only Input/Output survive, :171-175); the prose (:165, :177) says:
order the vertices of the mode by degree, assign them to the kappa partitions, order the hyperedges by partition id.
DESIGN.md reading 3: descending degree, each vertex to the currently least-loaded partition, ties to the lowest
partition id and the lowest vertex index - the longest-first rule whose worst case is the 4/3 (- 1/(3 kappa)) bound
the paper cites (:181).  Pins (tests/test_partition.py): the Fig. 2 example (:179: degrees 2, 1, 1 and kappa = 2 give
loads 2 and 2), the bound against the brute-force optimum on small inputs, and conservation of the load.
"""
from itertools import product


def partition_rows(degrees, kappa):
    """Returns (part_of_row, loads)."""
    order = sorted(range(len(degrees)), key=lambda v: (-degrees[v], v))
    loads = [0] * kappa
    part = [0] * len(degrees)
    for v in order:
        z = min(range(kappa), key=lambda b: (loads[b], b))
        part[v] = z
        loads[z] += degrees[v]
    return part, loads


def optimal_makespan(degrees, kappa):
    """Brute force over all assignments (tiny inputs only)."""
    best = None
    for assign in product(range(kappa), repeat=len(degrees)):
        loads = [0] * kappa
        for v, z in enumerate(assign):
            loads[z] += degrees[v]
        m = max(loads)
        best = m if best is None else min(best, m)
    return best
