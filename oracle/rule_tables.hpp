// ORACLE — TEST INFRASTRUCTURE ONLY.  Not part of the product path; shares no code with the
// CUDA library under paper_1606_03743_b200/csrc (which carries its own, independently typed
// transcription of the same tables).
//
// The ten Gaussian cubature rules of arXiv 1606.03743, Appendix A (triangles, barycentric
// coordinates) and Appendix B (rectangles, natural coordinates in
// [-1,1]^2), expanded to full point lists in long double.
// Rule summary PAPER.md L125: triangles (N,d) = (4,3) (7,5) (12,7) (19,9) (33,12);
// rectangles (N,d) = (4,3) (7,5) (12,7) (17,9) (33,13).
//
// Order of the expanded points: table row order; inside a row the permutations in the order
// the table caption lists them (cyclic for A3, "all different permutations" in lexicographic
// order of the position of the distinguished coordinate for the others).  The order only
// affects rounding.
//
// Readings of garbled table cells:
//  * A2 row 2 is blank in PAPER.md L297; taken from the caption L292 and the worked example
//    L127: (t+2ts, t-ts, t-ts) with weight (155+sqrt15)/1200; row 3 = (t+2tr, t-tr, t-tr)
//    with weight (155-sqrt15)/1200.
//  * B1-B3 print "S"/"-S" for s: lower-case symbols of the captions, all sign changes.
//  * A1's negative centroid weight -9/16 is kept as printed (L287).
#pragma once
#include <cmath>
#include <vector>

namespace orc {

typedef long double real;

struct TriNode  { real la, lb, lc, w; };
struct RectNode { real x, y, w; };

inline void tri_centroid(std::vector<TriNode>& v, real w) {
    v.push_back({1.0L / 3.0L, 1.0L / 3.0L, 1.0L / 3.0L, w});
}
// (a,b,b): the three different permutations ("like rows two to four in Table A1")
inline void tri_perm3(std::vector<TriNode>& v, real a, real b, real w) {
    v.push_back({a, b, b, w});
    v.push_back({b, a, b, w});
    v.push_back({b, b, a, w});
}
// cyclic permutations: (A,B,C) -> (B,C,A) -> (C,A,B)
inline void tri_cyc3(std::vector<TriNode>& v, real a, real b, real c, real w) {
    v.push_back({a, b, c, w});
    v.push_back({b, c, a, w});
    v.push_back({c, a, b, w});
}
// all six permutations
inline void tri_perm6(std::vector<TriNode>& v, real a, real b, real c, real w) {
    v.push_back({a, b, c, w});
    v.push_back({a, c, b, w});
    v.push_back({b, a, c, w});
    v.push_back({b, c, a, w});
    v.push_back({c, a, b, w});
    v.push_back({c, b, a, w});
}

// level 0..4 -> Tables A1..A5
inline std::vector<TriNode> tri_rule(int level) {
    std::vector<TriNode> v;
    switch (level) {
    case 0: {  // Table A1, N=4, degree 3 (L283-290)
        tri_centroid(v, -9.0L / 16.0L);
        tri_perm3(v, 3.0L / 5.0L, 1.0L / 5.0L, 25.0L / 48.0L);
        break;
    }
    case 1: {  // Table A2, N=7, degree 5 (L292-298)
        const real s15 = sqrtl(15.0L);
        const real t = 1.0L / 3.0L, s = (1.0L - s15) / 7.0L, r = (1.0L + s15) / 7.0L;
        tri_centroid(v, 9.0L / 40.0L);
        tri_perm3(v, t + 2.0L * t * s, t - t * s, (155.0L + s15) / 1200.0L);
        tri_perm3(v, t + 2.0L * t * r, t - t * r, (155.0L - s15) / 1200.0L);
        break;
    }
    case 2: {  // Table A3, N=12, degree 7 (L300-307)
        tri_cyc3(v, 0.06238226509439084L, 0.06751786707392436L, 0.8700998678316848L, 0.05303405631486900L);
        tri_cyc3(v, 0.05522545665692000L, 0.3215024938520156L, 0.6232720494910644L, 0.08776281742889622L);
        tri_cyc3(v, 0.03432430294509488L, 0.6609491961867980L, 0.3047265008681072L, 0.05755008556995056L);
        tri_cyc3(v, 0.5158423343536001L, 0.2777161669764050L, 0.2064414986699949L, 0.13498637401961758L);
        break;
    }
    case 3: {  // Table A4, N=19, degree 9 (L309-318)
        tri_centroid(v, 0.09713579628279610L);
        tri_perm3(v, 0.02063496160252593L, 0.48968251919873704L, 0.03133470022713983L);
        tri_perm3(v, 0.1258208170141290L, 0.4370895914929355L, 0.07782754100477543L);
        tri_perm3(v, 0.6235929287619356L, 0.18820353561903219L, 0.07964773892720910L);
        tri_perm3(v, 0.9105409732110941L, 0.04472951339445297L, 0.02557767565869810L);
        tri_perm6(v, 0.03683841205473626L, 0.7411985987844980L, 0.22196298916076573L, 0.04328353937728940L);
        break;
    }
    case 4: {  // Table A5, N=33, degree 12 (L320-331)
        tri_perm3(v, 0.4570749859701478L, 0.27146250701492611L, 0.06254121319590276L);
        tri_perm3(v, 0.1197767026828138L, 0.44011164865859310L, 0.04991833492806094L);
        tri_perm3(v, 0.0235924981089169L, 0.48820375094554155L, 0.02426683808145203L);
        tri_perm3(v, 0.7814843446812914L, 0.10925782765935432L, 0.02848605206887754L);
        tri_perm3(v, 0.9507072731273288L, 0.02464636343633558L, 0.00793164250997364L);
        tri_perm6(v, 0.1162960196779266L, 0.2554542286385173L, 0.62824975168355610L, 0.04322736365941421L);
        tri_perm6(v, 0.02303415635526714L, 0.2916556797383410L, 0.68531016390639186L, 0.02178358503860756L);
        tri_perm6(v, 0.02138249025617059L, 0.1272797172335894L, 0.85133779251024000L, 0.01508367757651144L);
        break;
    }
    default: break;
    }
    return v;
}

// all sign changes of (x,y), x,y != 0
inline void rect_signs4(std::vector<RectNode>& v, real x, real y, real w) {
    v.push_back({x, y, w});
    v.push_back({x, -y, w});
    v.push_back({-x, y, w});
    v.push_back({-x, -y, w});
}
// rotations by 0, 180, +-90 degrees: (x,y), (-x,-y), (-y,x), (y,-x)
inline void rect_rot4(std::vector<RectNode>& v, real x, real y, real w) {
    v.push_back({x, y, w});
    v.push_back({-x, -y, w});
    v.push_back({-y, x, w});
    v.push_back({y, -x, w});
}

// level 0..4 -> Tables B1..B5
inline std::vector<RectNode> rect_rule(int level) {
    std::vector<RectNode> v;
    switch (level) {
    case 0: {  // Table B1, N=4, degree 3 (L335-342)
        const real s = 1.0L / sqrtl(3.0L);
        rect_signs4(v, s, s, 0.25L);
        break;
    }
    case 1: {  // Table B2, N=7, degree 5 (L344-351)
        const real t = sqrtl(14.0L / 15.0L), r = sqrtl(3.0L / 5.0L), s = sqrtl(1.0L / 3.0L);
        v.push_back({0.0L, 0.0L, 2.0L / 7.0L});
        v.push_back({0.0L, t, 5.0L / 63.0L});
        v.push_back({0.0L, -t, 5.0L / 63.0L});
        rect_signs4(v, r, s, 5.0L / 36.0L);
        break;
    }
    case 2: {  // Table B3, N=12, degree 7 (L353-362)
        const real q583 = sqrtl(583.0L);
        const real r = sqrtl(6.0L / 7.0L);
        const real s = sqrtl((114.0L - 3.0L * q583) / 287.0L);
        const real t = sqrtl((114.0L + 3.0L * q583) / 287.0L);
        const real B1 = 49.0L / 810.0L;
        const real B2 = (178981.0L + 2769.0L * q583) / 1888920.0L;
        const real B3 = (178981.0L - 2769.0L * q583) / 1888920.0L;
        v.push_back({r, 0.0L, B1});
        v.push_back({-r, 0.0L, B1});
        v.push_back({0.0L, r, B1});
        v.push_back({0.0L, -r, B1});
        rect_signs4(v, s, s, B2);
        rect_signs4(v, t, t, B3);
        break;
    }
    case 3: {  // Table B4, N=17, degree 9 (L364-372)
        v.push_back({0.0L, 0.0L, 0.131687242798353921L});
        rect_rot4(v, 0.968849966361977720L, 0.630680119731668854L, 0.022219844542549678L);
        rect_rot4(v, 0.750277099978900533L, 0.927961645959569667L, 0.028024900532399120L);
        rect_rot4(v, 0.523735820214429336L, 0.453339821135647190L, 0.099570609815517519L);
        rect_rot4(v, 0.076208328192617173L, 0.852615729333662307L, 0.067262834409945196L);
        break;
    }
    case 4: {  // Table B5, N=33, degree 13 (L374-386)
        v.push_back({0.0L, 0.0L, 0.075095528857806335L});
        rect_rot4(v, 0.778809711554419422L, 0.983486682439872263L, 0.007497959716124783L);
        rect_rot4(v, 0.957297699786307365L, 0.859556005641638928L, 0.009543605329270918L);
        rect_rot4(v, 0.138183459862465353L, 0.958925170287534857L, 0.015106230954437494L);
        rect_rot4(v, 0.941327225872925236L, 0.390736216129461000L, 0.019373184633276336L);
        rect_rot4(v, 0.475808625218275905L, 0.850076673699748575L, 0.029711166825148901L);
        rect_rot4(v, 0.755805356572081436L, 0.647821637187010732L, 0.032440887592500675L);
        rect_rot4(v, 0.696250078491749413L, 0.070741508996444936L, 0.053335395364297350L);
        rect_rot4(v, 0.342716556040406789L, 0.409304561694038843L, 0.064217687370491966L);
        break;
    }
    default: break;
    }
    return v;
}

inline int tri_degree(int level)  { static const int d[5] = {3, 5, 7, 9, 12}; return d[level]; }
inline int rect_degree(int level) { static const int d[5] = {3, 5, 7, 9, 13}; return d[level]; }

}  // namespace orc
