"""Hand-worked block moves of the paper's main redistribution algorithm, shared by the oracle pins (tests/test_oracle_pins.py)
and the pins of the product's host plan (tests/test_dist_gloo.py).  No code: the expected counts below were written out by hand."""
# Hand-worked moves of the paper's main algorithm (A6b, reading G21: the block goes from the
# largest excess to the largest shortage, ties on EITHER side -> lowest index).  The cases are chosen so that the rule for
# equal excesses decides the final counts: an odd number of moves is shared among the tied partitions.
# (born, B, maxexc, counts, moves); r = balanced counts, e = cnt - r, window W = maxexc * B
MAIN_BY_HAND = [
    # r = (30,30,30), e = (10,10,-20): only the shortage is outside W = 10; one move, from partition 0 (not 1): e = (0,10,-10)
    ([40, 40, 10], 10, 1, [30, 40, 20], 1),
    # r = 30 x 4, e = (10,10,10,-30): 0->3 e = (0,10,10,-20); tie of 1 and 2 -> 1->3 e = (0,0,10,-10): stop
    ([40, 40, 40, 0], 10, 1, [30, 30, 40, 20], 2),
    # the tie appears only after the first move: e = (20,10,-30): 0->2 e = (10,10,-20); tie -> 0->2 e = (0,10,-10): stop
    ([50, 40, 0], 10, 1, [30, 40, 20], 2),
    # remainder: R' = 91, r = (31,30,30), e = (10,11,-21): 1->2 e = (10,1,-11); 0->2 e = (0,1,-1): stop
    ([41, 41, 9], 10, 1, [31, 31, 29], 2),
    # equal excesses AND equal shortages, even number of moves (either tie rule ends here; the moves are 0->2, 1->3)
    ([50, 50, 10, 10], 10, 1, [40, 40, 20, 20], 2),
    # window of two blocks: R' = 135, r = 45 x 3, e = (15,15,-30), W = 20: one move, from partition 0: e = (5,15,-20): stop
    ([60, 60, 15], 10, 2, [50, 60, 25], 1),
    # blocks of one replica: r = 10 x 3, e = (2,2,-4), W = 1: 0->2 (1,2,-3); 1->2 (1,1,-2); tie -> 0->2 (0,1,-1): stop
    ([12, 12, 6], 1, 1, [10, 11, 9], 3),
]
