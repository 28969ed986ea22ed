"""CPU oracle for the motion-focus hot path (TEST INFRASTRUCTURE, not product).

Plain, slow, fp64 restatement of what the path computes, written from
/root/reference/PAPER.md (cited as P:NN) and BASELINE.json's north_star (BJ).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference leg may import this package.  It shares no code with
paper_2601_07154_b200/ and never imports it.

Modules
  attention.py  softmax(QK^T/sqrt(D))V, global and per-frame      (BJ north_star)
  windows.py    sliding-window partition
  chain.py      incremental anchoring / pose chaining
  points.py     Eq. 1-6 motion points and the focus pixel
  render.py     Eq. 7 focus map and motion-guided depth
  block.py      linear / GELU / LayerNorm around the attention    (reading E1-E4)
  depth.py      depth scale on the window overlap, stream stitching (reading F2)

Parity status: every function is pinned by
tests/test_oracle_*.py except the *choices* the paper leaves open, which are
"parity unpinned" by the paper itself: B2 (which shared frame anchors),
C6 (CURRENT_FRAME vs OWN_FRAME aggregation), D1 (Z = max vs sum) and
D2 (guided depth = M*D); the block structure E1-E4 of block.py is a reading of BJ's
"d=1024 H=16 stack" (the paper names no block); F1 (bilinear depth upsampling) and F2 (least-squares
depth scale on the overlap) are readings of steps the paper is silent on.
"""
