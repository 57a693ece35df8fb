"""S6 track-candidate lists ("Each track candidate is a list of spacepoints"; line 89:
the service's output is the track candidates; line 184 "proto-track").  SURVEY.md section 8(f) NEXT-1.

Input: the S5 labels (label[v] = smallest hit index of v's component) and a minimum number of hits.
A track candidate is a component with at least `min_hits` hits.  The output is unique:

    tracks are ordered by their label (= their smallest hit index), ascending;
    the hits of a track are listed in ascending hit index;
    track_offsets int32 [T+1] (offsets[0] = 0), track_hits int32 [offsets[T]].

Hits of smaller components (noise, fragments) appear in no track.  The paper does not state a
minimum length; it is a hyperparameter here (reading C-23), 3 by default in the tests:
three hits is the least that fixes a helix.

Written as the definition: a dictionary of lists filled in index order.  Pure Python, O(N).
"""
from __future__ import annotations

import numpy as np


def build_tracks(labels, min_hits):
    labels = np.asarray(labels).astype(np.int64).tolist()
    members = {}
    for v, lab in enumerate(labels):          # index order, so every list is ascending
        members.setdefault(lab, []).append(v)
    offsets = [0]
    hits = []
    for lab in sorted(members):               # tracks by ascending label
        m = members[lab]
        if len(m) >= max(int(min_hits), 1):
            hits.extend(m)
            offsets.append(len(hits))
    return np.asarray(offsets, dtype=np.int32), np.asarray(hits, dtype=np.int32)
