"""Hand-built little positions in which chases happen all the time: inputs
for the chasing-rule tests of the oracle and of the CUDA path.  Layout helpers only."""
from paper_2511_07312_b200 import workloads as W


def _adj(a, b):
    return abs(a // 10 - b // 10) + abs(a % 10 - b % 10) == 1


def crowded(rng):
    # six movable pieces a side on the files between and beside the lakes, rows 2..7
    squares = [r * 10 + q for r in range(2, 8) for q in (0, 1, 4, 5, 8, 9)]
    rng.shuffle(squares)
    pieces = {9: W.piece(W.FLAG, W.RED), 90: W.piece(W.FLAG, W.BLUE)}
    types = [W.CAPTAIN, W.SERGEANT, W.SCOUT, W.MINER, W.MAJOR, W.SCOUT]
    for i, t in enumerate(types):
        pieces[squares[i]] = W.piece(t, W.RED)
        pieces[squares[6 + i]] = W.piece(t, W.BLUE)
    return pieces


def cage(rng):
    # one movable piece a side inside a small cage walled by Bombs: positions recur all the time
    free = [11, 12, 13, 21, 22, 23] if rng.random() < 0.5 else [11, 12, 21, 22]
    wall = set()
    for c in free:
        for d in (10, -10, 1, -1):
            n = c + d
            if 0 <= n <= 99 and _adj(c, n) and n not in free:
                wall.add(n)
    pieces = {9: W.piece(W.FLAG, W.RED), 99: W.piece(W.FLAG, W.BLUE)}
    for n in wall:
        pieces[n] = W.piece(W.BOMB, W.RED if rng.random() < 0.5 else W.BLUE)
    a, b = rng.choice(len(free), 2, replace=False)
    kinds = [W.SCOUT, W.SERGEANT, W.CAPTAIN]
    pieces[free[a]] = W.piece(kinds[rng.integers(3)], W.RED)
    pieces[free[b]] = W.piece(kinds[rng.integers(3)], W.BLUE)
    return pieces


