"""Oracle: sliding-window partition ("overlapping segments of size L sharing
O frames"; "only the newly processed, non-overlapping frames are emitted").

Reading B6: when (N-W) is not a multiple of stride = W-O, the last
window starts at N-W (larger overlap) and emits only the remaining frames.
TEST INFRASTRUCTURE ONLY.
"""


def num_windows(num_frames, w, stride):
    assert num_frames >= w and 1 <= stride < w
    return -(-(num_frames - w) // stride) + 1          # ceil((N-W)/stride) + 1


def window_starts(num_frames, w, stride):
    return [min(n * stride, num_frames - w) for n in range(num_windows(num_frames, w, stride))]


def emitted(num_frames, w, stride):
    """Per window: (global_begin, global_end) of the frames it emits, half-open."""
    starts = window_starts(num_frames, w, stride)
    out = [(0, w)]
    for n in range(1, len(starts)):
        out.append((starts[n - 1] + w, starts[n] + w))
    return out


def owner_of_frames(num_frames, w, stride):
    """For every global frame t: (window n, local index k) that emits it."""
    starts = window_starts(num_frames, w, stride)
    owner = [None] * num_frames
    for n, (b, e) in enumerate(emitted(num_frames, w, stride)):
        for t in range(b, e):
            owner[t] = (n, t - starts[n])
    assert all(o is not None for o in owner)
    return owner
