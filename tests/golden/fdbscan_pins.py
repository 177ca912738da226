"""Hand-worked FDBSCAN point sets (reading K-ii of DESIGN.md section 3), shared by the oracle pins
(tests/test_oracle_next.py) and the product-side checks (tests/test_candidates_host.py).  Data only: no arithmetic of the method.

Coordinates are small integers (time, DM); the SNR of every point is 10.  q is a neighbour of p when |dt| <= EPS and
|dDM| <= EPS (p included); a core point has >= min_pts neighbours.  Every expected label list and query count below was
worked out BY HAND from the paper's sentence "the representative points are chosen to be at the border of a core point's
neighborhood, two for each dimension, one for each direction when placing the core point at the origin" read as: per
dimension and direction, the neighbour OF THIS CLUSTER farthest from the core point (strictly positive displacement,
the lowest index among equals), each point expanded at most once, breadth first.  The walk-through of each set is in
the comment above it; `fails_for` names the one-line misreading the set is built to expose.
"""

# SPLIT -- "in some cases clusters might be split apart".  eps = 8, min_pts = 4.
#   0 A (0,0) with its four border points 1 (8,0), 2 (-8,0), 3 (0,8), 4 (0,-8) and an inner neighbour 5 q (7,7);
#   6..9 a tight group (14,14), (15,15), (14,15), (15,14) that only q reaches (q-6: 7,7; q-7: 8,8; 1-6: dDM 14).
#   A: neighbours {0..5}, all labelled 0; representatives +t 1 (8 > q's 7), -t 2, +DM 3 (8 > 7), -DM 4: q is none of them.
#   1: {0,1,3,4,5} core; +t none, -t 0/3/4 tie at 8 -> 0 (expanded), +DM 3, -DM 4.   2: {0,2,3,4} core, nothing new.
#   3: {0,1,2,3,5} core; +t 1, -t 2, -DM 0: all expanded.   4: {0,1,2,4} core, nothing new.   5 queries so far.
#   q is never expanded, although it is a core point ({0,1,3,5,6,7,8,9}): DBSCAN chains all ten points into ONE cluster.
#   Outer loop reaches 6: {5,6,7,8,9} core -> cluster 1 (q keeps label 0); +t 7/9 tie at 1 -> 7, +DM 7/8 tie -> 7.
#   7: {5,6,7,8,9} core; -t 6/8 tie -> 6 (expanded), -DM 6/9 -> 6.   7 queries in all.
SPLIT = dict(
    pts=[(0, 0), (8, 0), (-8, 0), (0, 8), (0, -8), (7, 7), (14, 14), (15, 15), (14, 15), (15, 14)],
    eps=8, min_pts=4,
    fdbscan_labels=[0, 0, 0, 0, 0, 0, 1, 1, 1, 1], fdbscan_queries=7,
    dbscan_labels=[0] * 10,
    fails_for="nearest instead of farthest representative (q, 7 away, would be A's +t seed: one cluster); no split at all",
)

# LOST -- "some points might be lost", and the tie-break.  eps = 8, min_pts = 4.
#   0 P (0,0); 1 r1 (8,-4) and 2 r2 (8,4) are equally far in +t; 5 (0,6) is the +DM border point; 3 (16,10), 4 (16,12) are
#   border points that only r2 reaches (r2: {0,1,2,3,4,5} core; r1: {0,1,2}; 5: {0,2,5}; 3: {2,3,4}; 4: {2,3,4}).
#   P: {0,1,2,5} core; +t r1/r2 tie at 8 -> the lower index r1; -t none; +DM 5 (6 > r2's 4); -DM r1.  r2 is not a seed.
#   r1 and 5 are not core points.  3 queries.  Outer loop: 3 and 4 have 3 neighbours each -> noise.  5 queries in all.
#   DBSCAN expands r2 and gives 3 and 4 to the cluster.
LOST = dict(
    pts=[(0, 0), (8, -4), (8, 4), (16, 10), (16, 12), (0, 6)],
    eps=8, min_pts=4,
    fdbscan_labels=[0, 0, 0, -1, -1, 0], fdbscan_queries=5,
    dbscan_labels=[0] * 6,
    fails_for="ties broken towards the higher index (r2 becomes the +t seed and brings 3 and 4 in)",
)

# OTHER -- representatives are taken among the neighbours "of this cluster".  eps = 4, min_pts = 4.
#   Cluster 0: 0 a0 (40,-4), 1 a1 (42,-4), 2 a2 (41,-2), 3 a3 (41,-6) and its border point 4 X (46,-1) (X: {1,4,5}, not core).
#   Cluster 1: 5 Q (50,3), 6 Y (48,6), 7 U (50,7), 8 Z (44,6).  Q: {4,5,6,7} core.  Seen from Q the farthest neighbour in -t is
#   X (4 away), but X belongs to cluster 0; the farthest OF THIS CLUSTER is Y (2 away).  Y: {5,6,7,8} core and the only
#   point that reaches Z; U: {5,6,7} is not core.
#   a0: {0,1,2,3}; +t a1, +DM a2, -DM a3.  a1: {0,1,2,3,4} labels X; +t X, +DM X, rest expanded/queued.  a2, a3: core, nothing
#   new.  X: 3 neighbours.  5 queries.  Q seeds cluster 1: -t Y, +DM U (4 > Y's 3), -DM none of this cluster.
#   Y: labels Z; -t Z, +DM U.  U: not core.  Z: {6,8}.  9 queries in all.
OTHER = dict(
    pts=[(40, -4), (42, -4), (41, -2), (41, -6), (46, -1), (50, 3), (48, 6), (50, 7), (44, 6)],
    eps=4, min_pts=4,
    fdbscan_labels=[0, 0, 0, 0, 0, 1, 1, 1, 1], fdbscan_queries=9,
    dbscan_labels=[0, 0, 0, 0, 0, 1, 1, 1, 1],
    fails_for="representatives drawn from ALL neighbours (X, already expanded, takes Q's -t slot; Y is never expanded, Z becomes noise)",
)

SETS = {"split": SPLIT, "lost": LOST, "other": OTHER}

# CHAIN -- a row of 7 points two apart along one axis, eps = 5, min_pts = 3: each expansion reaches two points further, and
# only the representative at the far end is expanded: points 0, 2, 4, 6 in the order met -> 4 queries, one cluster.
# Along time, DM or SNR, ascending or descending: six cases, one per (dimension, direction) of the paper's sentence.
CHAIN = dict(n=7, step=2, eps=5, min_pts=3, fdbscan_queries=4,
             fails_for="a dimension or direction without representative (the chain breaks into several clusters); nearest "
                       "representative (7 queries)")
